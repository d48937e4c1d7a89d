// api.cu -- the C ABI of include/lqcd.h: context, argument checks, the composition of
// Mhat / Mhat^dag from two hopping launches with fused epilogues, and the CG driver.
//
// Mhat(mu)     = M_ee - D_eo M_oo^{-1} D_oe                     (reading G3)
// Mhat(mu)^dag = M_ee^dag - D_eo^adj (M_oo^{-1})^dag D_oe^adj   (adjoint stencil, c -> -c)
// with c = 2 kappa mu, M = 1 + i c gamma5, M^{-1} = (1 - i c gamma5)/(1 + c^2), so per
// chirality chi = +-1 the diagonal terms are the complex numbers (1 + i c chi) and
// (1 - i c chi)/(1 + c^2); they are folded into the hopping kernel's epilogue:
//   launch 1: t   = [-kappa (1 - i c chi)/(1 + c^2)] * bracket(in)          (odd sites)
//   launch 2: out = kappa * (bracket(t) + [(1 + i c chi)/kappa] in)        (even sites)
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "../../include/lqcd.h"
#include "lqcd_internal.h"

#include <cstdint>

namespace lqcd {

static std::atomic<long long> g_launches{0};
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
// Programmatic dependent launches (lqcd_internal.h) for launches that go straight into the stream.  Not while the
// stream is being captured, by the library's own CG graph or by the caller: inside a graph the kernels already follow
// each other at ~2 us, and programmatic edges there measured neutral (24^3 x 48 and up) to 8-13% slower (16^4).
static bool g_prof_on = false;
// ... and not while lqcd_profile records an event pair around every launch: a chained kernel starts inside the pair of
// the kernel before it and the per-launch durations stop meaning what bench.py's roofline figure takes them for.
bool chained_launches(cudaStream_t st) {
    static const bool on = !(getenv("LQCD_PDL") && atoi(getenv("LQCD_PDL")) == 0);
    if (!on || g_prof_on) return false;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { cudaGetLastError(); return false; }
    return cs == cudaStreamCaptureStatusNone;
}

// ---- per-launch event timing (off by default; bench.py turns it on for the roofline figure)
struct ProfRec { int cat; cudaEvent_t a, b; };
static std::vector<ProfRec> g_prof;
static std::vector<cudaEvent_t> g_prof_pool;
static cudaEvent_t prof_event() {
    cudaEvent_t e = nullptr;
    if (!g_prof_pool.empty()) { e = g_prof_pool.back(); g_prof_pool.pop_back(); }
    else cudaEventCreate(&e);
    return e;
}
static void prof_clear() {
    for (auto& r : g_prof) { g_prof_pool.push_back(r.a); g_prof_pool.push_back(r.b); }
    g_prof.clear();
}
void prof_begin(int category, cudaStream_t st) {
    if (!g_prof_on) return;
    ProfRec r; r.cat = category; r.a = prof_event(); r.b = prof_event();
    cudaEventRecord(r.a, st);
    g_prof.push_back(r);
}
void prof_end(cudaStream_t st) {
    if (!g_prof_on || g_prof.empty()) return;
    cudaEventRecord(g_prof.back().b, st);
}

namespace {

struct Context {
    bool init = false;
    int dims[4] = {0, 0, 0, 0};
    Geometry geo;
    int precision = LQCD_DOUBLE;
    int recon = 18;
    int block = 128;
    cudaStream_t stream = 0;
    int snake = 1;                   // direction of the last field-sized launch (next_reverse)

    // workspace (owned), one set of half spinors per precision: r, p, q, t1, t2, t3
    void* vec[2][6] = {{nullptr, nullptr, nullptr, nullptr, nullptr, nullptr},
                       {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr}};
    void* full_b[2] = {nullptr, nullptr};  // lqcd_solve_full: right-hand side of the normal equations
    void* mx_b = nullptr;            // mixed solver: single-precision right-hand side and correction
    void* mx_x = nullptr;
    CgScalars* scal = nullptr;       // scalars of the running CG
    // four CG iterations as one instantiated CUDA graph, kept while the arguments it was captured with stay the same
    struct CgGraph {
        cudaGraphExec_t exec = nullptr;
        // the key: every argument of the 28 captured launches, and the stream the capture was tried on
        bool keyed = false;          // the fields below describe a capture attempt (exec != null: it worked)
        cudaStream_t stream = nullptr;
        int kind = 0;                // 0: CG on Mhat^dag Mhat (enqueue_iteration), 1: BiCGStab on Mhat (enqueue_bicg_iteration)
        const void* gauge = nullptr; void* x = nullptr; const void* b = nullptr;   // b: BiCGStab's rhat
        void* vec[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
        double* partials = nullptr; const void* scal = nullptr;
        int prec = -1, recon = 0, block = 0, launches = 0;
        double kappa = 0.0, mu = 0.0;
    } cgg;
    CgScalars* scal_outer = nullptr; // scalars of the mixed solver's outer (double) loop
    BiScalars* bscal = nullptr;      // scalars of the running BiCGStab
    CgScalars* scal_host = nullptr;  // pinned, 3 slots
    cudaEvent_t ev[2] = {nullptr, nullptr};
    double* partials = nullptr;
    size_t n_partials = 0;

    // host-call staging (owned)
    void* st_gauge_canon = nullptr; size_t st_gauge_canon_bytes = 0;
    void* st_gauge = nullptr;       size_t st_gauge_bytes = 0;
    void* st_spinor_canon = nullptr; size_t st_spinor_canon_bytes = 0;
    void* st_in = nullptr;  size_t st_in_bytes = 0;
    void* st_out = nullptr; size_t st_out_bytes = 0;

    // current solve
    int cg_prec = 0, cg_recon = 18;
    const void* cg_gauge = nullptr;
    const void* cg_b = nullptr;
    void* cg_x = nullptr;
    double cg_kappa = 0, cg_mu = 0, cg_tol = 0;
    bool cg_active = false;
    int st_iters = 0, st_outer = 0;
    double st_rr = 0, st_rt = 0;

    // slab decomposition (lqcd_slab_init): this rank's slab of the time direction
    bool slab = false;
    int rank = 0, nranks = 1;
    int s3 = 0;                      // sites per time slice and parity
    double* slab_sum = nullptr;      // the rank's partial sum awaiting the caller's all-reduce
};

// lqcd_select_context switches between independent contexts (lattice, format, stream, workspace,
// solver state): one per slab when several ranks of a slab decomposition share a process (tests).
constexpr int MAX_CONTEXTS = 8;
Context g_ctx[MAX_CONTEXTS];
int g_cur = 0;
#define ctx (g_ctx[g_cur])
char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int cuda_fail(cudaError_t e, const char* what) {
    return fail(LQCD_CUDA_ERROR, "%s: %s", what, cudaGetErrorString(e));
}

#define CU(call)                                                  \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);       \
    } while (0)

// sizes of the grouped layout: G groups of 32 sites per parity (pad sites included)
size_t spinor_bytes_of(int precision, int G) { return (size_t)G * 32 * 12 * (precision == 0 ? 16 : 8); }
size_t gauge_bytes_of(int precision, int recon, int G) {
    return (size_t)G * 32 * 8 * recon * (precision == 0 ? 8 : 4);
}
size_t n_reals() { return (size_t)24 * 32 * ctx.geo.G; }  // reals in one half-spinor field

void drop_cg_graph() {
    if (ctx.cgg.exec) cudaGraphExecDestroy(ctx.cgg.exec);
    ctx.cgg = Context::CgGraph();
}

void free_workspace() {
    drop_cg_graph();     // its launches hold the workspace pointers
    for (int pr = 0; pr < 2; ++pr)
        for (int i = 0; i < 6; ++i) { if (ctx.vec[pr][i]) cudaFree(ctx.vec[pr][i]); ctx.vec[pr][i] = nullptr; }
    for (int pr = 0; pr < 2; ++pr) { if (ctx.full_b[pr]) cudaFree(ctx.full_b[pr]); ctx.full_b[pr] = nullptr; }
    if (ctx.mx_b) cudaFree(ctx.mx_b);
    if (ctx.mx_x) cudaFree(ctx.mx_x);
    ctx.mx_b = ctx.mx_x = nullptr;
}

void free_all() {
    free_workspace();
    if (ctx.scal) cudaFree(ctx.scal);
    if (ctx.scal_outer) cudaFree(ctx.scal_outer);
    if (ctx.bscal) cudaFree(ctx.bscal);
    if (ctx.scal_host) cudaFreeHost(ctx.scal_host);
    if (ctx.partials) cudaFree(ctx.partials);
    if (ctx.slab_sum) cudaFree(ctx.slab_sum);
    for (int i = 0; i < 2; ++i) if (ctx.ev[i]) cudaEventDestroy(ctx.ev[i]);
    void** st[] = {&ctx.st_gauge_canon, &ctx.st_gauge, &ctx.st_spinor_canon, &ctx.st_in, &ctx.st_out};
    for (void** p : st) { if (*p) cudaFree(*p); *p = nullptr; }
    ctx = Context();
}

int ensure_scalars() {
    if (!ctx.scal) {
        CU(cudaMalloc(&ctx.scal, sizeof(CgScalars)));
        CU(cudaMemset(ctx.scal, 0, sizeof(CgScalars)));
        CU(cudaMalloc(&ctx.scal_outer, sizeof(CgScalars)));
        CU(cudaMemset(ctx.scal_outer, 0, sizeof(CgScalars)));
        CU(cudaMalloc(&ctx.bscal, sizeof(BiScalars)));
        CU(cudaMemset(ctx.bscal, 0, sizeof(BiScalars)));
        CU(cudaMallocHost(&ctx.scal_host, 3 * sizeof(CgScalars)));
        for (int i = 0; i < 2; ++i) CU(cudaEventCreateWithFlags(&ctx.ev[i], cudaEventDisableTiming));
    }
    // one partial per warp of a hopping launch, or up to three per block of a vector kernel (BiCGStab)
    // (a BiCGStab hopping launch leaves up to five sets of per-warp partials)
    size_t need = 5 * (size_t)hopping_partials(ctx.geo.Vh, 32) + 3 * (size_t)vector_grid(n_reals()) + 64;
    if (need < (size_t)plaquette_partials(ctx.geo.Vh)) need = (size_t)plaquette_partials(ctx.geo.Vh);
    if (need > ctx.n_partials) {
        drop_cg_graph();
        if (ctx.partials) CU(cudaFree(ctx.partials));
        ctx.partials = nullptr;
        CU(cudaMalloc(&ctx.partials, need * sizeof(double)));
        ctx.n_partials = need;
    }
    return LQCD_OK;
}

int ensure_workspace(int precision, int nvec) {
    int rc = ensure_scalars();
    if (rc) return rc;
    const size_t sb = spinor_bytes_of(precision, ctx.geo.Gg);
    // t1 (index 3) is needed by lqcd_mtm; the rest only by the solvers (t3 only by BiCGStab)
    const int order[6] = {3, 4, 0, 1, 2, 5};
    for (int k = 0; k < nvec; ++k) {
        const int i = order[k];
        if (!ctx.vec[precision][i]) CU(cudaMalloc(&ctx.vec[precision][i], sb));
    }
    return LQCD_OK;
}

int ensure_buf(void** p, size_t* have, size_t need) {
    if (*have >= need) return LQCD_OK;
    if (*p) CU(cudaFree(*p));
    *p = nullptr; *have = 0;
    CU(cudaMalloc(p, need));
    *have = need;
    return LQCD_OK;
}

Reduction red() { Reduction r; r.partials = ctx.partials; return r; }

int check_scalar(double v, const char* name) {
    if (!std::isfinite(v)) return fail(LQCD_BAD_ARG, "%s is not finite", name);
    return LQCD_OK;
}

// Snake order (lqcd_internal.h): every field-sized launch of a chain traverses the sites in the
// direction opposite to the launch before it.
int next_reverse() { return ctx.snake ^= 1; }

// The first hopping launch of Mhat (dagger = 0) or Mhat^dag (dagger = 1): even -> odd,
//   out_odd = M_oo^-1 D_oe in           (dagger = 0)
//   out_odd = (M_oo^-1)^dag (D_eo)^dag in   (dagger = 1; adjoint stencil, c -> -c)
int hop_minv(int precision, int recon, const void* gauge, const void* in, void* out_odd, double kappa,
             double mu, int dagger, CgScalars* scal) {
    const double c = (dagger ? -1.0 : 1.0) * 2.0 * kappa * mu;
    const double d = 1.0 + c * c;
    Epilogue e1 = {};
    e1.cu_re = -kappa / d; e1.cu_im = +kappa * c / d;   // -kappa (1 - i c)/(1 + c^2), chi = +1
    e1.cd_re = -kappa / d; e1.cd_im = -kappa * c / d;   // chi = -1
    CU(launch_hopping(precision, recon, dagger, 0, ctx.geo, e1, gauge, in, out_odd, nullptr, 1,
                      next_reverse(), red(), scal, ctx.block, ctx.stream));
    return LQCD_OK;
}

// The two hopping launches of Mhat (dagger = 0) or Mhat^dag (dagger = 1) on even half fields.
// fuse = FUSE_PAP: also reduce |out|^2 into scal->pAp (CG's <p, A p> = |Mhat p|^2).
// fuse = FUSE_R:   `out` is CG's residual r; instead of storing Mhat^(dag) in, the second launch
//                  applies r -= alpha * (Mhat^(dag) in) in place and reduces |r|^2 (FIN_RHO).
// scal: device scalars whose `done` flag turns the launches into no-ops (CG), or null.
// fuse = FUSE_DOT:  also leave the partial sums of |out|^2 and <dotw, out> (hopping.cu MODE 4; BiCGStab sums them).
enum { FUSE_NONE = 0, FUSE_PAP = 1, FUSE_R = 2, FUSE_DOT = 3 };
int apply_mhat(int precision, int recon, const void* gauge, const void* in, void* tmp_odd, void* out,
               double kappa, double mu, int dagger, int fuse, CgScalars* scal, const void* dotw = nullptr,
               const void* dotw2 = nullptr) {
    const double c = (dagger ? -1.0 : 1.0) * 2.0 * kappa * mu;
    int rc = hop_minv(precision, recon, gauge, in, tmp_odd, kappa, mu, dagger, scal);
    if (rc) return rc;
    // out = (1 + i c chi) in + kappa * bracket(t) = k2 * (bracket(t) + [(1 + i c chi)/k2] in).
    // For kappa = 0 launch 1 wrote t = 0 exactly, so bracket(t) = 0 and any k2 != 0 is exact.
    const double k2 = (kappa != 0.0) ? kappa : 1.0;
    Epilogue e2 = {};
    e2.cu_re = k2; e2.cd_re = k2;
    e2.du_re = 1.0 / k2; e2.du_im = c / k2;
    e2.dd_re = 1.0 / k2; e2.dd_im = -c / k2;
    e2.su_re = 1.0 / k2; e2.sd_re = 1.0 / k2;
    const int mode = (fuse == FUSE_PAP) ? 2 : (fuse == FUSE_R) ? 3 : (fuse == FUSE_DOT) ? (dotw2 ? 5 : 4) : 1;
    CU(launch_hopping(precision, recon, dagger, mode, ctx.geo, e2, gauge, tmp_odd,
                      out, in, 0, next_reverse(), red(), scal, ctx.block, ctx.stream, nullptr, dotw, dotw2));
    if (fuse == FUSE_PAP || fuse == FUSE_R)
        CU(launch_finalize(fuse == FUSE_PAP ? FIN_PAP : FIN_RHO, red(), hopping_partials(ctx.geo.Vh, ctx.block),
                           0.0, scal, ctx.stream));
    return LQCD_OK;
}

int enqueue_iteration() {
    void** v = ctx.vec[ctx.cg_prec];
    void *r = v[0], *p = v[1], *t1 = v[3], *t2 = v[4];
    const size_t n = n_reals();
    int rc = apply_mhat(ctx.cg_prec, ctx.cg_recon, ctx.cg_gauge, p, t1, t2, ctx.cg_kappa, ctx.cg_mu, 0, FUSE_PAP, ctx.scal);
    if (rc) return rc;
    // q = Mhat^dag t2 is never stored: the last hopping launch updates r in place (hopping.cu MODE 3)
    rc = apply_mhat(ctx.cg_prec, ctx.cg_recon, ctx.cg_gauge, t2, t1, r, ctx.cg_kappa, ctx.cg_mu, 1, FUSE_R, ctx.scal);
    if (rc) return rc;
    CU(launch_cg_update_xp(ctx.cg_prec, n, ctx.cg_x, p, r, next_reverse(), ctx.scal, ctx.stream));
    return LQCD_OK;
}

int cg_setup_impl(int precision, int recon, const void* gauge, const void* b, void* x, double kappa,
                  double mu, double tol) {
    int rc = ensure_workspace(precision, 5);
    if (rc) return rc;
    ctx.cg_prec = precision; ctx.cg_recon = recon;
    ctx.cg_gauge = gauge; ctx.cg_b = b; ctx.cg_x = x;
    ctx.cg_kappa = kappa; ctx.cg_mu = mu; ctx.cg_tol = tol;
    CU(launch_cg_init(precision, n_reals(), b, x, ctx.vec[precision][0], ctx.vec[precision][1],
                      tol, red(), ctx.scal, ctx.stream));
    ctx.cg_active = true;
    return LQCD_OK;
}

// One BiCGStab iteration on Mhat x = b (vector_ops.cu "BiCGStab"; rhat = b).
int enqueue_bicg_iteration() {
    void** w = ctx.vec[ctx.cg_prec];
    void *r = w[0], *p = w[1], *v = w[2], *t1 = w[3], *s = w[4], *t = w[5];
    const size_t n = n_reals();
    const int pr = ctx.cg_prec;
    CgScalars* gate = &ctx.bscal->cg;
    // sigma = <rhat, v> and <s, t>, |t|^2 come out of the hopping launches that produce v and t (MODE 4)
    const int G = ctx.geo.G;
    int rc = apply_mhat(pr, ctx.cg_recon, ctx.cg_gauge, p, t1, v, ctx.cg_kappa, ctx.cg_mu, 0, FUSE_DOT, gate, ctx.cg_b);
    if (rc) return rc;
    CU(launch_bicg_finalize(FIN_BI_SIGMA_HOP, red(), G, ctx.bscal, ctx.stream));
    CU(launch_bicg_s(pr, n, r, v, s, next_reverse(), ctx.bscal, ctx.stream));
    if ((rc = apply_mhat(pr, ctx.cg_recon, ctx.cg_gauge, s, t1, t, ctx.cg_kappa, ctx.cg_mu, 0, FUSE_DOT, gate, s, ctx.cg_b))) return rc;
    CU(launch_bicg_finalize(FIN_BI_OMEGA_BETA, red(), G, ctx.bscal, ctx.stream));
    CU(launch_bicg_xrp(pr, n, ctx.cg_x, p, s, t, v, r, next_reverse(), red(), ctx.bscal, ctx.stream));
    return LQCD_OK;
}

// Enqueue up to maxit iterations in chunks; the convergence flag of chunk k is read back while
// chunk k+1 is already queued, so the device never idles on the host.  `scal` is the solver's
// device scalar block (a CgScalars, or the CgScalars at the head of a BiScalars).
// The chunk of four CG iterations (28 launches; BiCGStab: 36) as one CUDA graph: between the kernels of a replayed graph
// the device loses ~1 us instead of the ~3 us of a stream launch, which is 18-27 us of the 63 / 113 us a CG
// iteration takes on 16^4 / 16^3 x 32 lattices.  Every argument of those launches is
// fixed during a solve (the scalars live on the device), so the graph is captured once and kept until one of
// the arguments changes.  Not used while per-launch events are recorded (lqcd_profile), in slab mode, when the
// caller is itself capturing the stream, or with LQCD_CG_GRAPH=0.
int enqueue_bicg_iteration();
bool cg_graph_ready(int kind = 0) {
    static const bool enabled = !(getenv("LQCD_CG_GRAPH") && atoi(getenv("LQCD_CG_GRAPH")) == 0);
    if (!enabled || g_prof_on || ctx.slab) return false;
    Context::CgGraph& c = ctx.cgg;
    void** v = ctx.vec[ctx.cg_prec];
    const void* scal = kind ? (const void*)ctx.bscal : (const void*)ctx.scal;
    const void* bkey = kind ? ctx.cg_b : nullptr;
    bool same = c.keyed && c.kind == kind && c.stream == ctx.stream && c.gauge == ctx.cg_gauge && c.x == ctx.cg_x && c.b == bkey &&
                c.prec == ctx.cg_prec && c.recon == ctx.cg_recon && c.block == ctx.block && c.kappa == ctx.cg_kappa &&
                c.mu == ctx.cg_mu && c.partials == ctx.partials && c.scal == scal;
    for (int i = 0; same && i < 6; ++i) same = (c.vec[i] == v[i]);
    // same arguments as the last attempt: replay its graph, or -- if the capture or the instantiation did not
    // work there (the legacy default stream cannot be captured) -- keep to direct launches without trying again
    if (same) return c.exec != nullptr;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(ctx.stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) { cudaGetLastError(); return false; }
    if (c.exec) { cudaGraphExecDestroy(c.exec); c.exec = nullptr; }
    c.keyed = true; c.kind = kind; c.stream = ctx.stream;
    c.gauge = ctx.cg_gauge; c.x = ctx.cg_x; c.b = bkey; c.prec = ctx.cg_prec; c.recon = ctx.cg_recon;
    c.block = ctx.block; c.kappa = ctx.cg_kappa; c.mu = ctx.cg_mu; c.partials = ctx.partials; c.scal = scal;
    for (int i = 0; i < 6; ++i) c.vec[i] = v[i];
    if (ctx.stream == 0 || ctx.stream == cudaStreamLegacy) return false;   // not capturable
    const long long l0 = g_launches.load();
    if (cudaStreamBeginCapture(ctx.stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return false; }
    int rc = 0;
    for (int i = 0; i < 4 && !rc; ++i) rc = kind ? enqueue_bicg_iteration() : enqueue_iteration();
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(ctx.stream, &graph);
    c.launches = (int)(g_launches.load() - l0);
    g_launches.store(l0);                       // nothing ran during the capture
    if (rc || e != cudaSuccess || !graph) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return false; }
    const cudaError_t ei = cudaGraphInstantiate(&c.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ei != cudaSuccess) { c.exec = nullptr; cudaGetLastError(); return false; }
    return true;
}

int cg_run_impl(int maxit, int (*enqueue)() = enqueue_iteration, const CgScalars* scal = nullptr) {
    if (!scal) scal = ctx.scal;
    const int chunk = 4;
    int launched = 0, slot = 0;
    bool pending[2] = {false, false};
    bool stop = false;
    while (launched < maxit && !stop) {
        const int n = (maxit - launched < chunk) ? (maxit - launched) : chunk;
        if (n == chunk && cg_graph_ready(enqueue == enqueue_iteration ? 0 : 1)) {
            CU(cudaGraphLaunch(ctx.cgg.exec, ctx.stream));
            count_launch(ctx.cgg.launches);
        } else {
            for (int i = 0; i < n; ++i) {
                int rc = enqueue();
                if (rc) return rc;
            }
        }
        launched += n;
        CU(cudaMemcpyAsync(&ctx.scal_host[slot], scal, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx.stream));
        CU(cudaEventRecord(ctx.ev[slot], ctx.stream));
        pending[slot] = true;
        const int prev = slot ^ 1;
        if (pending[prev]) {
            CU(cudaEventSynchronize(ctx.ev[prev]));
            pending[prev] = false;
            if (ctx.scal_host[prev].done) stop = true;
        }
        slot ^= 1;
    }
    return LQCD_OK;
}

// Synchronise; optionally compute the true residual |b - A x| (one more application of A with
// the `done` gate off); fill the statistics; return the solve status.
int cg_finish_stats(bool true_resid);
int cg_finish_impl(bool true_resid) {
    void** v = ctx.vec[ctx.cg_prec];
    if (true_resid) {
        void *q = v[2], *t1 = v[3], *t2 = v[4];
        int rc = apply_mhat(ctx.cg_prec, ctx.cg_recon, ctx.cg_gauge, ctx.cg_x, t1, t2, ctx.cg_kappa, ctx.cg_mu, 0, FUSE_NONE, nullptr);
        if (rc) return rc;
        rc = apply_mhat(ctx.cg_prec, ctx.cg_recon, ctx.cg_gauge, t2, t1, q, ctx.cg_kappa, ctx.cg_mu, 1, FUSE_NONE, nullptr);
        if (rc) return rc;
        CU(launch_true_resid(ctx.cg_prec, n_reals(), ctx.cg_b, q, red(), ctx.scal, ctx.stream));
    }
    return cg_finish_stats(true_resid);
}

// Synchronise, fill the statistics of lqcd_cg_stats from the device scalars, return the solve status.
int cg_finish_stats(bool true_resid) {
    CU(cudaMemcpyAsync(ctx.scal_host, ctx.scal, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx.stream));
    CU(cudaStreamSynchronize(ctx.stream));
    const CgScalars& s = ctx.scal_host[0];
    ctx.st_iters = s.iters;
    ctx.st_outer = 0;
    ctx.st_rr = s.bb > 0 ? std::sqrt(s.rho / s.bb) : 0.0;
    ctx.st_rt = (true_resid && s.bb > 0) ? std::sqrt(s.resid_true / s.bb) : 0.0;
    ctx.cg_active = false;
    if (s.status == LQCD_BREAKDOWN) return fail(LQCD_BREAKDOWN, "CG breakdown: <p,Ap> = %g", s.pAp);
    return s.status;
}

}  // namespace
}  // namespace lqcd

using namespace lqcd;

extern "C" {

const char* lqcd_last_error(void) { return g_err; }

int lqcd_init(const int dims[4], const double bc_phase[8]) {
    if (!dims || !bc_phase) return fail(LQCD_BAD_ARG, "lqcd_init: null argument");
    long long V = 1;
    for (int m = 0; m < 4; ++m) {
        if (dims[m] < 2 || (dims[m] & 1)) return fail(LQCD_BAD_DIMS, "extent %d = %d must be even and >= 2", m, dims[m]);
        V *= dims[m];
        const double a = std::hypot(bc_phase[2 * m], bc_phase[2 * m + 1]);
        if (!std::isfinite(a) || std::fabs(a - 1.0) > 1e-12)
            return fail(LQCD_BAD_DIMS, "|bc_phase[%d]| = %g must be 1", m, a);
    }
    if (V / 2 > (1LL << 30)) return fail(LQCD_BAD_DIMS, "lattice too large for 32-bit site indices");
    if (ctx.init) free_all();
    ctx.init = true;
    for (int m = 0; m < 4; ++m) {
        ctx.dims[m] = dims[m];
        ctx.geo.ph_re[m] = bc_phase[2 * m];
        ctx.geo.ph_im[m] = bc_phase[2 * m + 1];
    }
    ctx.geo.real_ph = 1;
    for (int m = 0; m < 4; ++m)
        if (bc_phase[2 * m + 1] != 0.0) ctx.geo.real_ph = 0;
    ctx.geo.N0h = dims[0] / 2; ctx.geo.N1 = dims[1]; ctx.geo.N2 = dims[2]; ctx.geo.N3 = dims[3];
    ctx.geo.d0h = make_fastdiv((unsigned)ctx.geo.N0h);
    ctx.geo.d1 = make_fastdiv((unsigned)ctx.geo.N1);
    ctx.geo.d2 = make_fastdiv((unsigned)ctx.geo.N2);
    ctx.geo.Vh = (int)(V / 2);
    ctx.geo.G = (ctx.geo.Vh + 31) / 32;
    ctx.geo.Gg = ctx.geo.G;
    ctx.s3 = ctx.geo.N0h * ctx.geo.N1 * ctx.geo.N2;
    ctx.geo.tph_f = ctx.geo.tph_b = 1;
    ctx.geo.slab = 0;
    ctx.slab = false; ctx.rank = 0; ctx.nranks = 1;
    ctx.precision = LQCD_DOUBLE; ctx.recon = 18; ctx.block = LQCD_DEFAULT_BLOCK; ctx.stream = 0;
    g_launches.store(0);
    g_err[0] = 0;
    return LQCD_OK;
}

int lqcd_finalize(void) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "lqcd_finalize: not initialised");
    cudaDeviceSynchronize();
    free_all();
    return LQCD_OK;
}

int lqcd_set_stream(void* cuda_stream) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    ctx.stream = (cudaStream_t)cuda_stream;
    return LQCD_OK;
}

int lqcd_set_format(int precision, int recon) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (precision != LQCD_DOUBLE && precision != LQCD_SINGLE) return fail(LQCD_BAD_ARG, "precision must be 0 or 1");
    if (recon != 18 && recon != 12) return fail(LQCD_BAD_ARG, "recon must be 18 or 12");
    ctx.precision = precision; ctx.recon = recon; ctx.cg_active = false;
    return LQCD_OK;
}

int lqcd_set_block_size(int threads) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (threads == 0) threads = LQCD_DEFAULT_BLOCK;
    if (threads < 32 || threads > LQCD_HOP_MAX_THREADS || (threads % 32)) return fail(LQCD_BAD_ARG, "block size must be 32, 64, 96 or 128");
    ctx.block = threads;
    return LQCD_OK;
}

int lqcd_set_hop_variant(int variant) {
    if (variant < 0 || variant > LQCD_HOP_VARIANT_MAX) return fail(LQCD_BAD_ARG, "hopping-kernel variant must be 0..%d", LQCD_HOP_VARIANT_MAX);
    for (int i = 0; i < MAX_CONTEXTS; ++i) {   // a captured CG chunk holds the kernels of the variant it was captured with
        if (g_ctx[i].cgg.exec) cudaGraphExecDestroy(g_ctx[i].cgg.exec);
        g_ctx[i].cgg = Context::CgGraph();
    }
    set_hopping_variant(variant);
    return LQCD_OK;
}

size_t lqcd_gauge_bytes(void) { return ctx.init ? gauge_bytes_of(ctx.precision, ctx.recon, ctx.geo.Gg) : 0; }
size_t lqcd_spinor_bytes(void) { return ctx.init ? spinor_bytes_of(ctx.precision, ctx.geo.Gg) : 0; }
long long lqcd_launch_count(void) { return g_launches.load(); }

int lqcd_profile(int enable) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (enable == 1) { CU(cudaStreamSynchronize(ctx.stream)); prof_clear(); }   // 2 = resume: keep the records, no sync
    g_prof_on = enable != 0;
    return LQCD_OK;
}

int lqcd_profile_read(int category, double* total_ms, int* launches) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    CU(cudaStreamSynchronize(ctx.stream));
    double tot = 0.0; int n = 0;
    for (const auto& r : g_prof) {
        if (r.cat != category) continue;
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, r.a, r.b));
        tot += ms; ++n;
    }
    if (total_ms) *total_ms = tot;
    if (launches) *launches = n;
    return LQCD_OK;
}

int lqcd_pack_gauge(const void* canon_dev, void* internal_dev) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (!canon_dev || !internal_dev) return fail(LQCD_BAD_ARG, "lqcd_pack_gauge: null pointer");
    CU(launch_pack_gauge(ctx.precision, ctx.recon, ctx.geo, canon_dev, internal_dev, ctx.stream));
    return LQCD_OK;
}

int lqcd_unpack_gauge(const void* internal_dev, void* canon_dev) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (!canon_dev || !internal_dev) return fail(LQCD_BAD_ARG, "lqcd_unpack_gauge: null pointer");
    CU(launch_unpack_gauge(ctx.precision, ctx.recon, ctx.geo, internal_dev, canon_dev, ctx.stream));
    return LQCD_OK;
}

// ---- the paper's copy micro-benchmark (stream_probe.cu; Fig. 5)
int lqcd_stream_probe(int elem, int mode, const void* src_dev, void* dst_dev, size_t bytes) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    static_assert(LQCD_STREAM_PROBE_BLOCKS == kStreamProbeBlocks, "header and kernel disagree on the READ grid");
    if (elem < LQCD_ELEM_FLOAT || elem > LQCD_ELEM_SPINOR_AOS) return fail(LQCD_BAD_ARG, "lqcd_stream_probe: elem must be 0..4");
    if (mode < LQCD_STREAM_COPY || mode > LQCD_STREAM_MIX71) return fail(LQCD_BAD_ARG, "lqcd_stream_probe: mode must be 0..2");
    if (elem >= LQCD_ELEM_SU3_AOS && mode != LQCD_STREAM_COPY) return fail(LQCD_BAD_ARG, "lqcd_stream_probe: the AoS elements support COPY only");
    if (bytes == 0) return LQCD_OK;
    if (!src_dev || !dst_dev) return fail(LQCD_BAD_ARG, "lqcd_stream_probe: null pointer");
    if (((uintptr_t)src_dev | (uintptr_t)dst_dev) & 15) return fail(LQCD_BAD_ARG, "lqcd_stream_probe: pointers must be 16-byte aligned");
    const size_t unit = (elem == LQCD_ELEM_SU3_AOS) ? 144 : (elem == LQCD_ELEM_SPINOR_AOS) ? 192 : (mode == LQCD_STREAM_MIX71) ? 112 : 16;
    if (bytes % unit) return fail(LQCD_BAD_ARG, "lqcd_stream_probe: bytes must be a multiple of 16 (144 / 192 for the AoS elements, 112 in MIX71)");
    CU(launch_stream_probe(elem, mode, src_dev, dst_dev, bytes, ctx.stream));
    return LQCD_OK;
}

int lqcd_fp64_probe(double a, double b, int iters, double* out_dev) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (!out_dev) return fail(LQCD_BAD_ARG, "lqcd_fp64_probe: null pointer");
    if (iters < 0) return fail(LQCD_BAD_ARG, "lqcd_fp64_probe: iters must be >= 0");
    int rc = check_scalar(a, "a");
    if (rc) return rc;
    rc = check_scalar(b, "b");
    if (rc) return rc;
    CU(launch_dfma_probe(a, b, iters, out_dev, ctx.stream));
    return LQCD_OK;
}

// ---- pure-gauge sector (gauge_update.cu): one launch per sub-sweep, 8 sub-sweeps per sweep
int lqcd_gauge_update(void* gauge, int mu, int parity, int mode, double beta, unsigned long long seed,
                      unsigned long long tag) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_gauge_update: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge) return fail(LQCD_BAD_ARG, "lqcd_gauge_update: null pointer");
    if (mu < 0 || mu > 3) return fail(LQCD_BAD_ARG, "mu must be 0..3");
    if (parity != 0 && parity != 1) return fail(LQCD_BAD_ARG, "parity must be 0 or 1");
    if (mode != LQCD_HEATBATH && mode != LQCD_OVERRELAX) return fail(LQCD_BAD_ARG, "mode must be LQCD_HEATBATH or LQCD_OVERRELAX");
    int rc = check_scalar(beta, "beta");
    if (rc) return rc;
    if (mode == LQCD_HEATBATH && !(beta > 0.0)) return fail(LQCD_BAD_ARG, "heatbath needs beta > 0");
    if (tag >= (1ull << 24)) return fail(LQCD_BAD_ARG, "tag must be below 2^24");
    // the heatbath's random-number counter reaches 1584 V (4 V links x 3 subgroups x 33 attempts x 4 draws) and
    // shares its 64-bit word with tag << 40 (reading G21): beyond 2^40 two tags would share numbers
    if (mode == LQCD_HEATBATH && 1584ull * 2ull * (unsigned long long)ctx.geo.Vh >= (1ull << 40))
        return fail(LQCD_BAD_DIMS, "heatbath: 1584 V = %llu random-number counters per sweep do not fit below 2^40",
                    1584ull * 2ull * (unsigned long long)ctx.geo.Vh);
    CU(launch_gauge_update(ctx.precision, ctx.recon, mode, ctx.geo, gauge, mu, parity, beta, seed, tag, ctx.stream));
    return LQCD_OK;
}

int lqcd_gauge_sweep(void* gauge, int mode, double beta, unsigned long long seed, unsigned long long tag) {
    for (int mu = 0; mu < 4; ++mu)
        for (int parity = 0; parity < 2; ++parity) {
            int rc = lqcd_gauge_update(gauge, mu, parity, mode, beta, seed, tag);
            if (rc) return rc;
        }
    return LQCD_OK;
}

int lqcd_plaquette(const void* gauge, double* plaquette_host) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_plaquette: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge || !plaquette_host) return fail(LQCD_BAD_ARG, "lqcd_plaquette: null pointer");
    int rc = ensure_scalars();
    if (rc) return rc;
    CU(launch_plaquette(ctx.precision, ctx.recon, ctx.geo, gauge, red(), ctx.stream));
    CU(launch_finalize(FIN_TRUE, red(), plaquette_partials(ctx.geo.Vh), 0.0, ctx.scal_outer, ctx.stream));
    CU(cudaMemcpyAsync(&ctx.scal_host[2], ctx.scal_outer, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx.stream));
    CU(cudaStreamSynchronize(ctx.stream));
    // sum of Re tr over the 6 V plaquettes -> average of Re tr / 3
    *plaquette_host = ctx.scal_host[2].resid_true / (3.0 * 6.0 * 2.0 * (double)ctx.geo.Vh);
    return LQCD_OK;
}

int lqcd_plaquette_static(const void* gauge, double* plaquette_dev) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_plaquette_static: not available after lqcd_slab_init");
    if (!gauge || !plaquette_dev) return fail(LQCD_BAD_ARG, "lqcd_plaquette_static: null pointer");
    const int np = plaquette_partials(ctx.geo.Vh);
    if (np > LQCD_PLAQUETTE_STATIC_MAX_PARTIALS)
        return fail(LQCD_BAD_ARG, "lqcd_plaquette_static: the lattice needs %d partial sums, the static scratch array holds %d "
                                  "(lattices up to 2^21 sites); use lqcd_plaquette", np, LQCD_PLAQUETTE_STATIC_MAX_PARTIALS);
    CU(launch_plaquette_static(ctx.precision, ctx.recon, ctx.geo, gauge, plaquette_dev, ctx.stream));
    return LQCD_OK;
}

int lqcd_pack_spinor(const void* canon_dev, void* internal_dev, int parity) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (!canon_dev || !internal_dev) return fail(LQCD_BAD_ARG, "lqcd_pack_spinor: null pointer");
    if (parity != 0 && parity != 1) return fail(LQCD_BAD_ARG, "parity must be 0 or 1");
    CU(launch_pack_spinor(ctx.precision, ctx.geo, canon_dev, internal_dev, parity, ctx.stream));
    return LQCD_OK;
}

int lqcd_unpack_spinor(const void* internal_dev, void* canon_dev, int parity) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (!canon_dev || !internal_dev) return fail(LQCD_BAD_ARG, "lqcd_unpack_spinor: null pointer");
    if (parity != 0 && parity != 1) return fail(LQCD_BAD_ARG, "parity must be 0 or 1");
    CU(launch_unpack_spinor(ctx.precision, ctx.geo, internal_dev, canon_dev, parity, ctx.stream));
    return LQCD_OK;
}

int lqcd_dslash_eo(const void* gauge, const void* in, void* out, int parity, double kappa) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (!gauge || !in || !out) return fail(LQCD_BAD_ARG, "lqcd_dslash_eo: null pointer");
    if (in == out) return fail(LQCD_BAD_ARG, "lqcd_dslash_eo: in and out alias");
    if (parity != 0 && parity != 1) return fail(LQCD_BAD_ARG, "parity must be 0 or 1");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    Epilogue ep = {};
    ep.cu_re = -kappa; ep.cd_re = -kappa;
    Reduction none = {nullptr};
    CU(launch_hopping(ctx.precision, ctx.recon, 0, 0, ctx.geo, ep, gauge, in, out, nullptr, parity, 0,
                      none, nullptr, ctx.block, ctx.stream));
    return LQCD_OK;
}

int lqcd_mtm(const void* gauge, const void* in, void* out, double kappa, double mu, int dagger) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_mtm: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge || !in || !out) return fail(LQCD_BAD_ARG, "lqcd_mtm: null pointer");
    if (in == out) return fail(LQCD_BAD_ARG, "lqcd_mtm: in and out alias");
    if (dagger != 0 && dagger != 1) return fail(LQCD_BAD_ARG, "dagger must be 0 or 1");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    rc = check_scalar(mu, "mu");
    if (rc) return rc;
    rc = ensure_workspace(ctx.precision, 1);
    if (rc) return rc;
    return apply_mhat(ctx.precision, ctx.recon, gauge, in, ctx.vec[ctx.precision][3], out, kappa, mu, dagger,
                      FUSE_NONE, nullptr);
}

// One hopping launch with the M_diag * aux epilogue: out_p = a_chi * (bracket(in) + d_chi aux).
static int hop_aux(const void* gauge, const void* in, const void* aux, void* out, int out_parity,
                   double cur, double cui, double cdr, double cdi, double dur, double dui, double ddr,
                   double ddi, int reverse) {
    Epilogue e = {};
    e.cu_re = cur; e.cu_im = cui; e.cd_re = cdr; e.cd_im = cdi;
    e.du_re = dur; e.du_im = dui; e.dd_re = ddr; e.dd_im = ddi;
    CU(launch_hopping(ctx.precision, ctx.recon, 0, 1, ctx.geo, e, gauge, in, out, aux, out_parity, reverse,
                      red(), nullptr, ctx.block, ctx.stream));
    return LQCD_OK;
}

int lqcd_mtm_full(const void* gauge, const void* in_even, const void* in_odd, void* out_even,
                  void* out_odd, double kappa, double mu) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_mtm_full: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge || !in_even || !in_odd || !out_even || !out_odd) return fail(LQCD_BAD_ARG, "lqcd_mtm_full: null pointer");
    if (out_even == in_even || out_even == in_odd || out_odd == in_even || out_odd == in_odd || out_even == out_odd)
        return fail(LQCD_BAD_ARG, "lqcd_mtm_full: buffers alias");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    if ((rc = check_scalar(mu, "mu"))) return rc;
    const double c = 2.0 * kappa * mu;
    if (kappa == 0.0) {  // M = M_diag
        CU(launch_diag_scale(ctx.precision, n_reals(), in_even, out_even, 1.0, c, 1.0, -c, ctx.stream));
        CU(launch_diag_scale(ctx.precision, n_reals(), in_odd, out_odd, 1.0, c, 1.0, -c, ctx.stream));
        return LQCD_OK;
    }
    // out_p = (1 + i c chi) in_p - kappa bracket(in_{1-p}) = -kappa (bracket + [(1 + i c chi)/(-kappa)] in_p)
    if ((rc = hop_aux(gauge, in_odd, in_even, out_even, 0, -kappa, 0, -kappa, 0, -1.0 / kappa, -c / kappa,
                      -1.0 / kappa, c / kappa, 0))) return rc;
    return hop_aux(gauge, in_even, in_odd, out_odd, 1, -kappa, 0, -kappa, 0, -1.0 / kappa, -c / kappa,
                   -1.0 / kappa, c / kappa, 1);
}

// M psi = eta on the whole lattice through the even-odd system:
//   rhs_e = eta_e - D_eo M_oo^{-1} eta_o;  Mhat^dag Mhat psi_e = Mhat^dag rhs_e (CG);
//   psi_o = M_oo^{-1} (eta_o - D_oe psi_e).
int lqcd_solve_full(const void* gauge, const void* eta_even, const void* eta_odd, void* psi_even,
                    void* psi_odd, double kappa, double mu, double tol, int maxit) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_solve_full: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge || !eta_even || !eta_odd || !psi_even || !psi_odd) return fail(LQCD_BAD_ARG, "lqcd_solve_full: null pointer");
    if (psi_even == eta_even || psi_even == eta_odd || psi_odd == eta_even || psi_odd == eta_odd || psi_even == psi_odd)
        return fail(LQCD_BAD_ARG, "lqcd_solve_full: buffers alias");
    if (maxit < 1) return fail(LQCD_BAD_ARG, "maxit must be >= 1");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    if ((rc = check_scalar(mu, "mu"))) return rc;
    if (!std::isfinite(tol) || tol < 0.0) return fail(LQCD_BAD_ARG, "tol must be finite and >= 0");
    const double c = 2.0 * kappa * mu, d = 1.0 + c * c;
    const size_t n = n_reals();
    if (kappa == 0.0) {  // M = M_diag: psi = M_diag^{-1} eta
        CU(launch_diag_scale(ctx.precision, n, eta_even, psi_even, 1.0 / d, -c / d, 1.0 / d, c / d, ctx.stream));
        CU(launch_diag_scale(ctx.precision, n, eta_odd, psi_odd, 1.0 / d, -c / d, 1.0 / d, c / d, ctx.stream));
        CU(cudaStreamSynchronize(ctx.stream));
        ctx.st_iters = 0; ctx.st_outer = 0; ctx.st_rr = ctx.st_rt = 0.0;
        return LQCD_OK;
    }
    if ((rc = ensure_workspace(ctx.precision, 5))) return rc;
    const int pr = ctx.precision;
    if (!ctx.full_b[pr]) CU(cudaMalloc(&ctx.full_b[pr], spinor_bytes_of(pr, ctx.geo.G)));
    // psi_even and psi_odd double as scratch until they receive their results
    CU(launch_diag_scale(pr, n, eta_odd, psi_even, 1.0 / d, -c / d, 1.0 / d, c / d, ctx.stream));   // u_o = M_oo^-1 eta_o
    if ((rc = hop_aux(gauge, psi_even, eta_even, psi_odd, 0, kappa, 0, kappa, 0, 1.0 / kappa, 0, 1.0 / kappa, 0, 1)))
        return rc;                                                                                  // rhs_e = eta_e - D_eo u_o
    if ((rc = apply_mhat(pr, ctx.recon, gauge, psi_odd, ctx.vec[pr][3], ctx.full_b[pr], kappa, mu, 1, FUSE_NONE, nullptr)))
        return rc;                                                                                  // b = Mhat^dag rhs_e
    if ((rc = cg_setup_impl(pr, ctx.recon, gauge, ctx.full_b[pr], psi_even, kappa, mu, tol))) return rc;
    if ((rc = cg_run_impl(maxit))) return rc;
    const int status = cg_finish_impl(true);
    if (status < 0) return status;
    // psi_o = M_oo^{-1} (eta_o - D_oe psi_e) = [kappa (1 - i c chi)/(1 + c^2)] (bracket(psi_e) + eta_o / kappa)
    if ((rc = hop_aux(gauge, psi_even, eta_odd, psi_odd, 1, kappa / d, -kappa * c / d, kappa / d, kappa * c / d,
                      1.0 / kappa, 0, 1.0 / kappa, 0, 0))) return rc;
    CU(cudaStreamSynchronize(ctx.stream));
    return status;
}

int lqcd_cg_setup(const void* gauge, const void* b, void* x, double kappa, double mu, double tol) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_cg_setup: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge || !b || !x) return fail(LQCD_BAD_ARG, "lqcd_cg_setup: null pointer");
    if (b == x) return fail(LQCD_BAD_ARG, "lqcd_cg_setup: b and x alias");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    rc = check_scalar(mu, "mu");
    if (rc) return rc;
    if (!std::isfinite(tol) || tol < 0.0) return fail(LQCD_BAD_ARG, "tol must be finite and >= 0");
    return cg_setup_impl(ctx.precision, ctx.recon, gauge, b, x, kappa, mu, tol);
}

int lqcd_cg_iterate(int n) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_cg_iterate: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!ctx.cg_active) return fail(LQCD_BAD_ARG, "lqcd_cg_iterate: no solve set up");
    if (n < 0) return fail(LQCD_BAD_ARG, "n must be >= 0");
    int i = 0;
    while (n - i >= 4 && cg_graph_ready()) {   // four iterations at a time as the cached graph (cg_run_impl)
        CU(cudaGraphLaunch(ctx.cgg.exec, ctx.stream));
        count_launch(ctx.cgg.launches);
        i += 4;
    }
    for (; i < n; ++i) {
        int rc = enqueue_iteration();
        if (rc) return rc;
    }
    return LQCD_OK;
}

int lqcd_cg_finish(void) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_cg_finish: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!ctx.cg_active) return fail(LQCD_BAD_ARG, "lqcd_cg_finish: no solve set up");
    return cg_finish_impl(true);
}

int lqcd_cg_mdagm(const void* gauge, const void* b, void* x, double kappa, double mu, double tol,
                  int maxit) {
    if (maxit < 1) return fail(LQCD_BAD_ARG, "maxit must be >= 1");
    int rc = lqcd_cg_setup(gauge, b, x, kappa, mu, tol);
    if (rc) return rc;
    rc = cg_run_impl(maxit);
    if (rc) return rc;
    return cg_finish_impl(true);
}

int lqcd_bicgstab_mhat(const void* gauge, const void* b, void* x, double kappa, double mu, double tol,
                       int maxit) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_bicgstab_mhat: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge || !b || !x) return fail(LQCD_BAD_ARG, "lqcd_bicgstab_mhat: null pointer");
    if (b == x) return fail(LQCD_BAD_ARG, "lqcd_bicgstab_mhat: b and x alias");
    if (maxit < 1) return fail(LQCD_BAD_ARG, "maxit must be >= 1");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    if ((rc = check_scalar(mu, "mu"))) return rc;
    if (!std::isfinite(tol) || tol < 0.0) return fail(LQCD_BAD_ARG, "tol must be finite and >= 0");
    const int pr = ctx.precision;
    if ((rc = ensure_workspace(pr, 6))) return rc;
    ctx.cg_prec = pr; ctx.cg_recon = ctx.recon;
    ctx.cg_gauge = gauge; ctx.cg_b = b; ctx.cg_x = x;
    ctx.cg_kappa = kappa; ctx.cg_mu = mu; ctx.cg_tol = tol;
    ctx.cg_active = false;   // the three-step CG interface is not open on this solve
    void** w = ctx.vec[pr];
    CU(launch_bicg_init(pr, n_reals(), b, x, w[0], w[1], tol, red(), ctx.bscal, ctx.stream));
    if ((rc = cg_run_impl(maxit, enqueue_bicg_iteration, &ctx.bscal->cg))) return rc;
    // true residual |b - Mhat x| / |b|
    if ((rc = apply_mhat(pr, ctx.recon, gauge, x, w[3], w[5], kappa, mu, 0, FUSE_NONE, nullptr))) return rc;
    CU(launch_true_resid(pr, n_reals(), b, w[5], red(), &ctx.bscal->cg, ctx.stream));
    CU(cudaMemcpyAsync(ctx.scal_host, &ctx.bscal->cg, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx.stream));
    CU(cudaStreamSynchronize(ctx.stream));
    const CgScalars& sc = ctx.scal_host[0];
    ctx.st_iters = sc.iters;
    ctx.st_outer = 0;
    ctx.st_rr = sc.bb > 0 ? std::sqrt(sc.rho / sc.bb) : 0.0;
    ctx.st_rt = sc.bb > 0 ? std::sqrt(sc.resid_true / sc.bb) : 0.0;
    if (sc.status == LQCD_BREAKDOWN) return fail(LQCD_BREAKDOWN, "BiCGStab breakdown after %d iterations", sc.iters);
    return sc.status;
}

size_t lqcd_force_bytes(void) { return ctx.init ? (size_t)ctx.geo.G * 32 * 2 * 4 * 8 * sizeof(double) : 0; }

int lqcd_unpack_force(const void* force_internal_dev, void* canon_dev) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (!force_internal_dev || !canon_dev) return fail(LQCD_BAD_ARG, "lqcd_unpack_force: null pointer");
    CU(launch_unpack_force(ctx.geo, force_internal_dev, canon_dev, ctx.stream));
    return LQCD_OK;
}

int lqcd_fermion_force(const void* gauge, const void* x_even, const void* x_odd, const void* y_even,
                       const void* y_odd, void* force, double kappa) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_fermion_force: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge || !x_even || !x_odd || !y_even || !y_odd || !force) return fail(LQCD_BAD_ARG, "lqcd_fermion_force: null pointer");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    CU(launch_fermion_force(ctx.precision, ctx.recon, ctx.geo, gauge, x_even, x_odd, y_even, y_odd, force, kappa,
                            ctx.stream));
    return LQCD_OK;
}

// Force of S = phi^dag (Mhat^dag Mhat)^-1 phi (reading G16):
//   X_e = (Mhat^dag Mhat)^-1 phi (CG);  Y_e = Mhat X_e, whose first hopping launch leaves
//   t1 = M_oo^-1 D_oe X_e = -X_o;  t2 = (M_oo^-1)^dag (D_eo)^dag Y_e = -Y_o (the first launch of
//   Mhat^dag on Y_e);  the common sign is handed to the force kernel as the sign of kappa.
int lqcd_force_tm(const void* gauge, const void* phi, void* force, double kappa, double mu, double tol,
                  int maxit) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_force_tm: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge || !phi || !force) return fail(LQCD_BAD_ARG, "lqcd_force_tm: null pointer");
    if (maxit < 1) return fail(LQCD_BAD_ARG, "maxit must be >= 1");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    if ((rc = check_scalar(mu, "mu"))) return rc;
    if (!std::isfinite(tol) || tol < 0.0) return fail(LQCD_BAD_ARG, "tol must be finite and >= 0");
    const int pr = ctx.precision;
    if ((rc = ensure_workspace(pr, 6))) return rc;
    void** w = ctx.vec[pr];
    void *ye = w[2], *t1 = w[3], *t2 = w[4], *xe = w[5];
    if ((rc = cg_setup_impl(pr, ctx.recon, gauge, phi, xe, kappa, mu, tol))) return rc;
    if ((rc = cg_run_impl(maxit))) return rc;
    const int status = cg_finish_impl(true);
    if (status < 0) return status;
    if ((rc = apply_mhat(pr, ctx.recon, gauge, xe, t1, ye, kappa, mu, 0, FUSE_NONE, nullptr))) return rc;
    if ((rc = hop_minv(pr, ctx.recon, gauge, ye, t2, kappa, mu, 1, nullptr))) return rc;
    // every term of the force holds exactly one odd-site field (X(x+mu) Y(x) or X(x) Y(x+mu) with x, x+mu of
    // opposite parity), so handing in t1 = -X_o and t2 = -Y_o flips the sign of the whole force: kappa -> -kappa
    CU(launch_fermion_force(pr, ctx.recon, ctx.geo, gauge, xe, t1, ye, t2, force, -kappa, ctx.stream));
    CU(cudaStreamSynchronize(ctx.stream));
    return status;
}

// Mixed-precision defect correction:
//   x = 0, r = b (double); repeat: solve A e = r/|r| in single by CG to inner_tol;
//   x += |r| e; r = b - A x in double; until |r| <= tol |b|.
int lqcd_cg_mdagm_mixed(const void* gauge_double, int recon_double, const void* gauge_single,
                        int recon_single, const void* b, void* x, double kappa, double mu, double tol,
                        int maxit, double inner_tol) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_cg_mdagm_mixed: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge_double || !gauge_single || !b || !x) return fail(LQCD_BAD_ARG, "lqcd_cg_mdagm_mixed: null pointer");
    if (b == x) return fail(LQCD_BAD_ARG, "lqcd_cg_mdagm_mixed: b and x alias");
    if ((recon_double != 18 && recon_double != 12) || (recon_single != 18 && recon_single != 12))
        return fail(LQCD_BAD_ARG, "recon must be 18 or 12");
    if (maxit < 1) return fail(LQCD_BAD_ARG, "maxit must be >= 1");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    if ((rc = check_scalar(mu, "mu"))) return rc;
    if (!std::isfinite(tol) || tol < 0.0) return fail(LQCD_BAD_ARG, "tol must be finite and >= 0");
    if (!std::isfinite(inner_tol) || inner_tol < 0.0 || inner_tol >= 1.0)
        return fail(LQCD_BAD_ARG, "inner_tol must be in [0, 1)");
    if ((rc = ensure_workspace(LQCD_DOUBLE, 5))) return rc;
    if ((rc = ensure_workspace(LQCD_SINGLE, 5))) return rc;
    const size_t sbf = spinor_bytes_of(LQCD_SINGLE, ctx.geo.G);
    if (!ctx.mx_b) CU(cudaMalloc(&ctx.mx_b, sbf));
    if (!ctx.mx_x) CU(cudaMalloc(&ctx.mx_x, sbf));
    void** vd = ctx.vec[LQCD_DOUBLE];
    void *r = vd[0], *q = vd[2], *t1 = vd[3], *t2 = vd[4];
    const size_t n = n_reals();
    CgScalars* so = ctx.scal_outer;
    CgScalars* sh = &ctx.scal_host[2];
    // x = 0, r = b, bb = rho = |b|^2 (p slot vd[1] is scratch here)
    CU(launch_cg_init(LQCD_DOUBLE, n, b, x, r, vd[1], tol, red(), so, ctx.stream));
    int total = 0, outer = 0, status = LQCD_NOT_CONVERGED;
    double rho = 0.0, bb = 0.0;
    for (;;) {
        CU(cudaMemcpyAsync(sh, so, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx.stream));
        CU(cudaStreamSynchronize(ctx.stream));
        bb = sh->bb;
        rho = (outer == 0) ? sh->rho : sh->resid_true;
        // NaN / inf first (a NaN in b or in the links, an overflow in the double residual): a NaN rho would
        // otherwise pass the negated convergence test below and be reported as converged
        if (!std::isfinite(rho) || !std::isfinite(bb)) { status = LQCD_BREAKDOWN; break; }
        if (!(rho > tol * tol * bb)) { status = LQCD_OK; break; }      // also catches b = 0
        if (total >= maxit) break;
        const double scale = std::sqrt(rho);
        CU(launch_convert_d2f(n, r, ctx.mx_b, 1.0 / scale, ctx.stream));
        // inner_tol = 0: ask each inner solve only for the reduction still missing (half of it,
        // for slack), but never for more than single precision delivers (1e-6)
        double itol = inner_tol;
        if (itol == 0.0) {
            itol = 0.5 * tol * std::sqrt(bb / rho);
            if (itol < 1e-6) itol = 1e-6;
            if (itol > 0.1) itol = 0.1;
        }
        rc = cg_setup_impl(LQCD_SINGLE, recon_single, gauge_single, ctx.mx_b, ctx.mx_x, kappa, mu, itol);
        if (rc) return rc;
        if ((rc = cg_run_impl(maxit - total))) return rc;
        const int ist = cg_finish_impl(false);
        if (ist < 0) return ist;
        total += ctx.st_iters;
        ++outer;
        CU(launch_axpy_f2d(n, scale, ctx.mx_x, x, ctx.stream));
        // r = b - A x in double
        if ((rc = apply_mhat(LQCD_DOUBLE, recon_double, gauge_double, x, t1, t2, kappa, mu, 0, FUSE_NONE, nullptr))) return rc;
        if ((rc = apply_mhat(LQCD_DOUBLE, recon_double, gauge_double, t2, t1, q, kappa, mu, 1, FUSE_NONE, nullptr))) return rc;
        CU(launch_residual(n, b, q, r, red(), so, ctx.stream));
        if (ctx.st_iters == 0) { status = LQCD_BREAKDOWN; break; }      // inner solver made no progress
    }
    ctx.st_iters = total;
    ctx.st_outer = outer;
    ctx.st_rr = ctx.st_rt = bb > 0 ? std::sqrt(rho / bb) : (std::isfinite(bb) ? 0.0 : bb);   // the outer residual IS a true residual
    ctx.cg_active = false;
    if (status == LQCD_BREAKDOWN) return fail(LQCD_BREAKDOWN, "mixed CG: no progress or not finite (|r|^2 = %g, |b|^2 = %g)", rho, bb);
    return status;
}

int lqcd_cg_outer_iterations(void) { return ctx.init ? ctx.st_outer : 0; }

int lqcd_cg_stats(int* iters, double* rel_resid_recursive, double* rel_resid_true) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (iters) *iters = ctx.st_iters;
    if (rel_resid_recursive) *rel_resid_recursive = ctx.st_rr;
    if (rel_resid_true) *rel_resid_true = ctx.st_rt;
    return LQCD_OK;
}

static int stage_inputs(const void* gauge_host, const void* spinor_host) {
    const size_t V = 2 * (size_t)ctx.geo.Vh;
    const size_t gc = V * 576, sc = (size_t)ctx.geo.Vh * 192;
    int rc;
    if ((rc = ensure_buf(&ctx.st_gauge_canon, &ctx.st_gauge_canon_bytes, gc))) return rc;
    if ((rc = ensure_buf(&ctx.st_gauge, &ctx.st_gauge_bytes, lqcd_gauge_bytes()))) return rc;
    if ((rc = ensure_buf(&ctx.st_spinor_canon, &ctx.st_spinor_canon_bytes, sc))) return rc;
    if ((rc = ensure_buf(&ctx.st_in, &ctx.st_in_bytes, lqcd_spinor_bytes()))) return rc;
    if ((rc = ensure_buf(&ctx.st_out, &ctx.st_out_bytes, lqcd_spinor_bytes()))) return rc;
    CU(cudaMemcpyAsync(ctx.st_gauge_canon, gauge_host, gc, cudaMemcpyHostToDevice, ctx.stream));
    CU(cudaMemcpyAsync(ctx.st_spinor_canon, spinor_host, sc, cudaMemcpyHostToDevice, ctx.stream));
    if ((rc = lqcd_pack_gauge(ctx.st_gauge_canon, ctx.st_gauge))) return rc;
    if ((rc = lqcd_pack_spinor(ctx.st_spinor_canon, ctx.st_in, 0))) return rc;
    return LQCD_OK;
}

static int fetch_output(void* out_host) {
    const size_t sc = (size_t)ctx.geo.Vh * 192;
    int rc = lqcd_unpack_spinor(ctx.st_out, ctx.st_spinor_canon, 0);
    if (rc) return rc;
    CU(cudaMemcpyAsync(out_host, ctx.st_spinor_canon, sc, cudaMemcpyDeviceToHost, ctx.stream));
    CU(cudaStreamSynchronize(ctx.stream));
    return LQCD_OK;
}

int lqcd_mtm_host(const void* gauge_canon_host, const void* in_canon_host, void* out_canon_host,
                  double kappa, double mu, int dagger) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_mtm_host: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge_canon_host || !in_canon_host || !out_canon_host) return fail(LQCD_BAD_ARG, "lqcd_mtm_host: null pointer");
    int rc = stage_inputs(gauge_canon_host, in_canon_host);
    if (rc) return rc;
    if ((rc = lqcd_mtm(ctx.st_gauge, ctx.st_in, ctx.st_out, kappa, mu, dagger))) return rc;
    return fetch_output(out_canon_host);
}

int lqcd_cg_mdagm_host(const void* gauge_canon_host, const void* b_canon_host, void* x_canon_host,
                       double kappa, double mu, double tol, int maxit) {
    if (!ctx.init) return fail(LQCD_NOT_INITIALISED, "not initialised");
    if (ctx.slab) return fail(LQCD_BAD_ARG, "lqcd_cg_mdagm_host: not available after lqcd_slab_init (use the lqcd_slab_* calls)");
    if (!gauge_canon_host || !b_canon_host || !x_canon_host) return fail(LQCD_BAD_ARG, "lqcd_cg_mdagm_host: null pointer");
    int rc = stage_inputs(gauge_canon_host, b_canon_host);
    if (rc) return rc;
    const int status = lqcd_cg_mdagm(ctx.st_gauge, ctx.st_in, ctx.st_out, kappa, mu, tol, maxit);
    if (status < 0) return status;
    rc = fetch_output(x_canon_host);
    return rc ? rc : status;
}

// ------------------------------------------------------------------------------------------------
// Slab decomposition of the time direction over several ranks, one GPU each (
// DESIGN.md section 7).  The library computes; the caller moves the halos and sums the scalars.
// ------------------------------------------------------------------------------------------------
int lqcd_select_context(int id) {
    if (id < 0 || id >= MAX_CONTEXTS) return fail(LQCD_BAD_ARG, "context id must be in [0, %d)", MAX_CONTEXTS);
    g_cur = id;
    return LQCD_OK;
}

int lqcd_slab_init(const int dims_global[4], const double bc_phase[8], int rank, int nranks) {
    if (!dims_global || !bc_phase) return fail(LQCD_BAD_ARG, "lqcd_slab_init: null argument");
    if (nranks < 1 || rank < 0 || rank >= nranks) return fail(LQCD_BAD_ARG, "rank %d of %d", rank, nranks);
    if (dims_global[3] % nranks) return fail(LQCD_BAD_DIMS, "N_t = %d is not a multiple of %d ranks", dims_global[3], nranks);
    int loc[4] = {dims_global[0], dims_global[1], dims_global[2], dims_global[3] / nranks};
    // the local extent must be even so that a site's parity in the slab equals its global parity
    int rc = lqcd_init(loc, bc_phase);
    if (rc) return rc;
    if (ctx.s3 % 32) {
        free_all();
        return fail(LQCD_BAD_DIMS, "slab mode needs N_x N_y N_z / 2 = %d sites per time slice and parity to be a multiple of 32",
                    (loc[0] / 2) * loc[1] * loc[2]);
    }
    ctx.slab = true; ctx.rank = rank; ctx.nranks = nranks;
    ctx.geo.slab = 1;
    ctx.geo.tph_f = (rank == nranks - 1);
    ctx.geo.tph_b = (rank == 0);
    ctx.geo.Gg = ctx.geo.G + 2 * (ctx.s3 / 32);
    return LQCD_OK;
}

static size_t site_bytes() { return spinor_bytes_of(ctx.precision, 1) / 32; }

int lqcd_slab_spinor_halo(size_t* send_lo, size_t* send_hi, size_t* ghost_fwd, size_t* ghost_bwd, size_t* bytes) {
    if (!ctx.init || !ctx.slab) return fail(LQCD_NOT_INITIALISED, "lqcd_slab_spinor_halo: no slab set up");
    const size_t sb = site_bytes(), Vh = ctx.geo.Vh, s3 = ctx.s3;
    if (send_lo) *send_lo = 0;
    if (send_hi) *send_hi = (Vh - s3) * sb;
    if (ghost_fwd) *ghost_fwd = Vh * sb;
    if (ghost_bwd) *ghost_bwd = (Vh + s3) * sb;
    if (bytes) *bytes = s3 * sb;
    return LQCD_OK;
}

int lqcd_slab_gauge_halo(int parity, size_t* send_hi, size_t* ghost_bwd, size_t* bytes) {
    if (!ctx.init || !ctx.slab) return fail(LQCD_NOT_INITIALISED, "lqcd_slab_gauge_halo: no slab set up");
    if (parity != 0 && parity != 1) return fail(LQCD_BAD_ARG, "parity must be 0 or 1");
    const size_t gb = (size_t)ctx.recon * 32 * (ctx.precision == 0 ? 8 : 4);   // bytes of one group of one (parity, mu) array
    const size_t base = ((size_t)(parity * 4 + 3) * ctx.geo.Gg) * gb;          // mu = 3
    if (send_hi) *send_hi = base + (size_t)((ctx.geo.Vh - ctx.s3) / 32) * gb;
    if (ghost_bwd) *ghost_bwd = base + (size_t)((ctx.geo.Vh + ctx.s3) / 32) * gb;
    if (bytes) *bytes = (size_t)(ctx.s3 / 32) * gb;
    return LQCD_OK;
}

// part: 0 every site, 1 interior time slices (no ghost needed), 2 the two boundary time slices
static int slab_range(int part, SiteRange* r) {
    const int Vh = ctx.geo.Vh, s3 = ctx.s3;
    const int inner = Vh - 2 * s3 > 0 ? Vh - 2 * s3 : 0;   // N3 = 2: every slice is a boundary slice
    if (part == 0) { r->base = 0; r->count = Vh; r->n1 = Vh; r->skip = 0; }
    else if (part == 1) { r->base = s3; r->count = inner; r->n1 = inner; r->skip = 0; }
    else if (part == 2) { r->base = 0; r->count = Vh - inner; r->n1 = s3; r->skip = inner; }
    else return fail(LQCD_BAD_ARG, "part must be 0 (all), 1 (interior) or 2 (boundary)");
    return LQCD_OK;
}

int lqcd_slab_dslash(const void* gauge, const void* in, void* out, int parity, double kappa, int part) {
    if (!ctx.init || !ctx.slab) return fail(LQCD_NOT_INITIALISED, "lqcd_slab_dslash: no slab set up");
    if (!gauge || !in || !out || in == out) return fail(LQCD_BAD_ARG, "lqcd_slab_dslash: null or aliased pointer");
    if (parity != 0 && parity != 1) return fail(LQCD_BAD_ARG, "parity must be 0 or 1");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    SiteRange rg;
    if ((rc = slab_range(part, &rg))) return rc;
    Epilogue ep = {};
    ep.cu_re = -kappa; ep.cd_re = -kappa;
    Reduction none = {nullptr};
    CU(launch_hopping(ctx.precision, ctx.recon, 0, 0, ctx.geo, ep, gauge, in, out, nullptr, parity, 0, none, nullptr,
                      ctx.block, ctx.stream, &rg));
    return LQCD_OK;
}

// One of the two hopping launches of Mhat / Mhat^dag (api.cu header), on the sites of `part`:
//   stage 1: tmp_odd = M_oo^-1 D_oe in          (needs the ghosts of `in`)
//   stage 2: out     = M_ee in - D_eo tmp_odd   (needs the ghosts of `tmp_odd`)
// fuse, scal as in apply_mhat (the sums stay partial: see slab_local_sum).
static int slab_mhat_stage(const void* gauge, const void* in, void* tmp_odd, void* out, double kappa, double mu,
                           int dagger, int stage, int part, int fuse, CgScalars* scal) {
    SiteRange rg;
    int rc = slab_range(part, &rg);
    if (rc) return rc;
    const double c = (dagger ? -1.0 : 1.0) * 2.0 * kappa * mu;
    if (stage == 1) {
        const double d = 1.0 + c * c;
        Epilogue e1 = {};
        e1.cu_re = -kappa / d; e1.cu_im = +kappa * c / d;
        e1.cd_re = -kappa / d; e1.cd_im = -kappa * c / d;
        CU(launch_hopping(ctx.precision, ctx.recon, dagger, 0, ctx.geo, e1, gauge, in, tmp_odd, nullptr, 1, 0, red(), scal,
                          ctx.block, ctx.stream, &rg));
    } else {
        const double k2 = (kappa != 0.0) ? kappa : 1.0;
        Epilogue e2 = {};
        e2.cu_re = k2; e2.cd_re = k2;
        e2.du_re = 1.0 / k2; e2.du_im = c / k2;
        e2.dd_re = 1.0 / k2; e2.dd_im = -c / k2;
        e2.su_re = 1.0 / k2; e2.sd_re = 1.0 / k2;
        const int mode = (fuse == FUSE_PAP) ? 2 : (fuse == FUSE_R) ? 3 : 1;
        CU(launch_hopping(ctx.precision, ctx.recon, dagger, mode, ctx.geo, e2, gauge, tmp_odd, out, in, 0, 0, red(), scal,
                          ctx.block, ctx.stream, &rg));
    }
    return LQCD_OK;
}

int lqcd_slab_mhat_stage(const void* gauge, const void* in, void* tmp_odd, void* out, double kappa, double mu,
                         int dagger, int stage, int part) {
    if (!ctx.init || !ctx.slab) return fail(LQCD_NOT_INITIALISED, "lqcd_slab_mhat_stage: no slab set up");
    if (!gauge || !in || !tmp_odd || !out || in == out || in == tmp_odd || tmp_odd == out)
        return fail(LQCD_BAD_ARG, "lqcd_slab_mhat_stage: null or aliased pointer");
    if ((dagger != 0 && dagger != 1) || (stage != 1 && stage != 2)) return fail(LQCD_BAD_ARG, "dagger must be 0 or 1, stage 1 or 2");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    if ((rc = check_scalar(mu, "mu"))) return rc;
    if ((rc = ensure_scalars())) return rc;
    return slab_mhat_stage(gauge, in, tmp_odd, out, kappa, mu, dagger, stage, part, FUSE_NONE, nullptr);
}

int lqcd_slab_cg_begin(const void* gauge, const void* b, void* x, double kappa, double mu, double tol) {
    if (!ctx.init || !ctx.slab) return fail(LQCD_NOT_INITIALISED, "lqcd_slab_cg_begin: no slab set up");
    if (!gauge || !b || !x || b == x) return fail(LQCD_BAD_ARG, "lqcd_slab_cg_begin: null or aliased pointer");
    int rc = check_scalar(kappa, "kappa");
    if (rc) return rc;
    if ((rc = check_scalar(mu, "mu"))) return rc;
    if (!std::isfinite(tol) || tol < 0.0) return fail(LQCD_BAD_ARG, "tol must be finite and >= 0");
    if ((rc = ensure_workspace(ctx.precision, 5))) return rc;
    if (!ctx.slab_sum) CU(cudaMalloc(&ctx.slab_sum, 2 * sizeof(double)));
    ctx.cg_prec = ctx.precision; ctx.cg_recon = ctx.recon;
    ctx.cg_gauge = gauge; ctx.cg_b = b; ctx.cg_x = x;
    ctx.cg_kappa = kappa; ctx.cg_mu = mu; ctx.cg_tol = tol;
    ctx.cg_active = true;
    return LQCD_OK;
}

void* lqcd_slab_sum_ptr(void) { return (ctx.init && ctx.slab) ? (void*)ctx.slab_sum : nullptr; }

// The field whose ghost slices stage `stage` reads (NULL: none).
void* lqcd_slab_cg_halo_field(int stage) {
    if (!ctx.init || !ctx.slab || !ctx.cg_active) return nullptr;
    void** v = ctx.vec[ctx.cg_prec];
    switch (stage) {
        case 2: return v[1];            // p
        case 3: case 7: case 12: case 14: return v[3];   // t1
        case 6: case 13: return v[4];   // t2
        case 11: return ctx.cg_x;
        default: return nullptr;
    }
}

int lqcd_slab_cg_stage(int stage, int part) {
    if (!ctx.init || !ctx.slab) return fail(LQCD_NOT_INITIALISED, "lqcd_slab_cg_stage: no slab set up");
    if (!ctx.cg_active) return fail(LQCD_BAD_ARG, "lqcd_slab_cg_stage: no solve set up (lqcd_slab_cg_begin)");
    void** v = ctx.vec[ctx.cg_prec];
    void *r = v[0], *p = v[1], *q = v[2], *t1 = v[3], *t2 = v[4];
    const size_t n = n_reals();
    const int np = hopping_partials(ctx.geo.Vh, ctx.block);
    const void* U = ctx.cg_gauge;
    const double ka = ctx.cg_kappa, mu = ctx.cg_mu;
    switch (stage) {
        case 0:   // r = p = b, x = 0, the rank's |b|^2
            CU(launch_cg_init(ctx.cg_prec, n, ctx.cg_b, ctx.cg_x, r, p, ctx.cg_tol, red(), ctx.scal, ctx.stream, ctx.slab_sum));
            return LQCD_OK;
        case 1: CU(launch_finalize(FIN_BB, red(), 0, ctx.cg_tol, ctx.scal, ctx.stream, ctx.slab_sum, 1)); return LQCD_OK;
        case 2: return slab_mhat_stage(U, p, t1, t2, ka, mu, 0, 1, part, FUSE_NONE, ctx.scal);
        case 3: return slab_mhat_stage(U, p, t1, t2, ka, mu, 0, 2, part, FUSE_PAP, ctx.scal);
        case 4: CU(launch_finalize(FIN_PAP, red(), np, 0.0, ctx.scal, ctx.stream, ctx.slab_sum, 0)); return LQCD_OK;
        case 5: CU(launch_finalize(FIN_PAP, red(), 0, 0.0, ctx.scal, ctx.stream, ctx.slab_sum, 1)); return LQCD_OK;
        case 6: return slab_mhat_stage(U, t2, t1, r, ka, mu, 1, 1, part, FUSE_NONE, ctx.scal);
        case 7: return slab_mhat_stage(U, t2, t1, r, ka, mu, 1, 2, part, FUSE_R, ctx.scal);
        case 8: CU(launch_finalize(FIN_RHO, red(), np, 0.0, ctx.scal, ctx.stream, ctx.slab_sum, 0)); return LQCD_OK;
        case 9:
            CU(launch_finalize(FIN_RHO, red(), 0, 0.0, ctx.scal, ctx.stream, ctx.slab_sum, 1));
            CU(launch_cg_update_xp(ctx.cg_prec, n, ctx.cg_x, p, r, 0, ctx.scal, ctx.stream));
            return LQCD_OK;
        // true residual |b - Mhat^dag Mhat x| (the `done` gate off)
        case 11: return slab_mhat_stage(U, ctx.cg_x, t1, t2, ka, mu, 0, 1, part, FUSE_NONE, nullptr);
        case 12: return slab_mhat_stage(U, ctx.cg_x, t1, t2, ka, mu, 0, 2, part, FUSE_NONE, nullptr);
        case 13: return slab_mhat_stage(U, t2, t1, q, ka, mu, 1, 1, part, FUSE_NONE, nullptr);
        case 14: return slab_mhat_stage(U, t2, t1, q, ka, mu, 1, 2, part, FUSE_NONE, nullptr);
        case 15: CU(launch_true_resid(ctx.cg_prec, n, ctx.cg_b, q, red(), ctx.scal, ctx.stream, ctx.slab_sum)); return LQCD_OK;
        case 16: CU(launch_finalize(FIN_TRUE, red(), 0, 0.0, ctx.scal, ctx.stream, ctx.slab_sum, 1)); return LQCD_OK;
        default: return fail(LQCD_BAD_ARG, "lqcd_slab_cg_stage: unknown stage %d", stage);
    }
}

// Synchronise and read the solver's scalars: *done = 1 once converged or broken down.
int lqcd_slab_cg_poll(int* done, int* iters) {
    if (!ctx.init || !ctx.slab || !ctx.cg_active) return fail(LQCD_BAD_ARG, "lqcd_slab_cg_poll: no solve set up");
    CgScalars s;
    CU(cudaMemcpyAsync(&ctx.scal_host[2], ctx.scal, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx.stream));
    CU(cudaStreamSynchronize(ctx.stream));
    s = ctx.scal_host[2];
    if (done) *done = s.done;
    if (iters) *iters = s.iters;
    return LQCD_OK;
}

int lqcd_slab_cg_end(int with_true_resid) { return (ctx.init && ctx.slab && ctx.cg_active) ? cg_finish_stats(with_true_resid != 0) : fail(LQCD_BAD_ARG, "lqcd_slab_cg_end: no solve set up"); }

}  // extern "C"
