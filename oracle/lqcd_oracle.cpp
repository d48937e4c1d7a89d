// lqcd_oracle.cpp -- TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, obviously-correct CPU statement of what the hot path computes:
// the twisted-mass Wilson fermion matrix of arxiv 1209.5942, eq. 6
// (PAPER.md:79-82), its even-odd blocks and Schur complement (named only at
// PAPER.md:94, :205, :223; reading G3 of DESIGN.md) and CG on M^dag M
// (eq. 8; reading G10).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may call this.  It shares no code, header, table or
// helper with the CUDA path under paper_1209_5942_b200/csrc and neither
// includes the other.  Arithmetic is std::complex<double>, compiled with
// -ffp-contract=off (reading G13); global sums accumulate in long double.
//
// There is no blocking, fusion or reordering here: every function is the
// definition written out, in the paper's notation, one output site at a time.
// (An OpenMP "parallel for" over independent output sites is the only
// concession to the timed baseline; it changes no arithmetic.)
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): free-field closed form (P1),
// gamma5-hermiticity and true adjointness (P2), gauge covariance (P3),
// entry-by-entry comparison with a dense 2^4 build written independently in
// numpy (P4), the paper's own identity M(mu)^dag M(mu) = M(0)^dag M(0) +
// 4 kappa^2 mu^2 (P5), Schur identity vs the dense matrix (P6),
// trivial limits (P7), CG vs a dense Hermitian solve (P8), BiCGStab vs a dense solve
// of Mhat and the textbook recurrence on the dense matrix (P9), the fermion force vs central
// differences of the action computed from dense matrices (P10).  The paper prints
// no numeric example for any of these operators, so element values rest on
// P1-P8.
//
// Canonical layout (row-major, complex = (re,im) doubles):
//   gauge   U[lex(x)][mu][a][b]           mu = 0..3 = x,y,z,t
//   spinor  psi[lex(x)][alpha][a]         alpha = Dirac 0..3, a = colour 0..2
//   half    psi_p[e][alpha][a]            e = lex(x)/2 over sites of parity p
//   lex(x) = x0 + N0*(x1 + N1*(x2 + N2*x3)),  parity(x) = (x0+x1+x2+x3) mod 2
// All extents even (>= 2), so lex 2k and 2k+1 have opposite parity and
// e = lex/2 is a bijection on each parity.

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <functional>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef std::complex<double> cplx;
const cplx I_(0.0, 1.0);
const cplx O_(0.0, 0.0);
const cplx E_(1.0, 0.0);

// ---------------------------------------------------------------------------
// gamma matrices.  The paper fixes only {gamma_mu, gamma_nu} = 2 delta_mu_nu
// (Euclidean).  Reading G4: the chiral basis of the paper's
// textbook reference [9]; gamma5 = gamma_x gamma_y gamma_z gamma_t
// = diag(1,1,-1,-1).  Rows listed top to bottom.
// ---------------------------------------------------------------------------
const cplx GAMMA[4][4][4] = {
    // gamma_x
    {{O_, O_, O_, -I_}, {O_, O_, -I_, O_}, {O_, I_, O_, O_}, {I_, O_, O_, O_}},
    // gamma_y
    {{O_, O_, O_, -E_}, {O_, O_, E_, O_}, {O_, E_, O_, O_}, {-E_, O_, O_, O_}},
    // gamma_z
    {{O_, O_, -I_, O_}, {O_, O_, O_, I_}, {I_, O_, O_, O_}, {O_, -I_, O_, O_}},
    // gamma_t
    {{O_, O_, E_, O_}, {O_, O_, O_, E_}, {E_, O_, O_, O_}, {O_, E_, O_, O_}},
};
const double GAMMA5[4] = {1.0, 1.0, -1.0, -1.0};

struct Lattice {
    int N[4];
    cplx phase[4];  // e^{i pi theta_mu}; applied on the hop that wraps (G5)
    long V;
};

Lattice make_lattice(const int* dims, const double* bc_phase) {
    Lattice L;
    L.V = 1;
    for (int m = 0; m < 4; ++m) {
        L.N[m] = dims[m];
        L.phase[m] = cplx(bc_phase[2 * m], bc_phase[2 * m + 1]);
        L.V *= dims[m];
    }
    return L;
}

long lex(const Lattice& L, const int* x) {
    return x[0] + (long)L.N[0] * (x[1] + (long)L.N[1] * (x[2] + (long)L.N[2] * x[3]));
}

void coords(const Lattice& L, long s, int* x) {
    x[0] = (int)(s % L.N[0]); s /= L.N[0];
    x[1] = (int)(s % L.N[1]); s /= L.N[1];
    x[2] = (int)(s % L.N[2]); s /= L.N[2];
    x[3] = (int)s;
}

int parity_of(const int* x) { return (x[0] + x[1] + x[2] + x[3]) & 1; }

// lex index of the e-th site of parity p: candidates 2e and 2e+1.
long lex_of_eo(const Lattice& L, long e, int p) {
    int x[4];
    coords(L, 2 * e, x);
    return (parity_of(x) == p) ? 2 * e : 2 * e + 1;
}

// A spinor field seen through an accessor: get(lex, out[12]).
typedef std::function<void(long, cplx*)> Field;

// (U psi)_{alpha,a} = sum_b U_ab psi_{alpha,b}
void su3_mul(const cplx* U, const cplx* psi, cplx* out) {
    for (int al = 0; al < 4; ++al)
        for (int a = 0; a < 3; ++a) {
            cplx s = O_;
            for (int b = 0; b < 3; ++b) s += U[3 * a + b] * psi[3 * al + b];
            out[3 * al + a] = s;
        }
}

// (U^dag psi)_{alpha,a} = sum_b conj(U_ba) psi_{alpha,b}
void su3_dag_mul(const cplx* U, const cplx* psi, cplx* out) {
    for (int al = 0; al < 4; ++al)
        for (int a = 0; a < 3; ++a) {
            cplx s = O_;
            for (int b = 0; b < 3; ++b) s += std::conj(U[3 * b + a]) * psi[3 * al + b];
            out[3 * al + a] = s;
        }
}

// out = (1 + sign * gamma_mu) v, the full 4x4 matrix acting on the Dirac index.
void one_plus_sgamma(int mu, double sign, const cplx* v, cplx* out) {
    for (int al = 0; al < 4; ++al)
        for (int a = 0; a < 3; ++a) {
            cplx s = v[3 * al + a];
            for (int be = 0; be < 4; ++be) s += sign * GAMMA[mu][al][be] * v[3 * be + a];
            out[3 * al + a] = s;
        }
}

// The bracket of eq. 6 at one site x (reading G1/G2: sum over the 8 signed
// directions, coefficient -kappa applied by the caller):
//   acc = sum_mu [ eta+_mu(x) (1 - s gamma_mu) U_mu(x)        psi(x+mu)
//                + eta-_mu(x) (1 + s gamma_mu) U_mu(x-mu)^dag psi(x-mu) ]
// s = +1 is eq. 6; s = -1 is the adjoint stencil (D^dag has gamma_mu -> -gamma_mu,
// same links, same phases).  eta+ = phase_mu if x_mu = N_mu-1, eta- =
// conj(phase_mu) if x_mu = 0, else 1 (G5).  For N_mu = 2 both hops reach the
// same site and both are added (G8).
void hop_site(const Lattice& L, const cplx* U, const Field& psi, const int* x, double s,
              cplx* acc) {
    for (int i = 0; i < 12; ++i) acc[i] = O_;
    const long sx = lex(L, x);
    cplx nb[12], t1[12], t2[12];
    for (int mu = 0; mu < 4; ++mu) {
        int y[4] = {x[0], x[1], x[2], x[3]};
        // forward hop
        y[mu] = (x[mu] + 1) % L.N[mu];
        cplx eta = (x[mu] == L.N[mu] - 1) ? L.phase[mu] : E_;
        psi(lex(L, y), nb);
        su3_mul(U + (sx * 4 + mu) * 9, nb, t1);
        one_plus_sgamma(mu, -s, t1, t2);
        for (int i = 0; i < 12; ++i) acc[i] += eta * t2[i];
        // backward hop
        y[mu] = (x[mu] + L.N[mu] - 1) % L.N[mu];
        eta = (x[mu] == 0) ? std::conj(L.phase[mu]) : E_;
        const long sy = lex(L, y);
        psi(sy, nb);
        su3_dag_mul(U + (sy * 4 + mu) * 9, nb, t1);
        one_plus_sgamma(mu, +s, t1, t2);
        for (int i = 0; i < 12; ++i) acc[i] += eta * t2[i];
    }
}

// M_diag^{+-} psi = (1 + i c gamma5) psi with c = 2 kappa mu (eq. 6); the
// adjoint has c -> -c.
void mdiag_site(double c, const cplx* v, cplx* out) {
    for (int al = 0; al < 4; ++al)
        for (int a = 0; a < 3; ++a)
            out[3 * al + a] = (E_ + I_ * (c * GAMMA5[al])) * v[3 * al + a];
}

// (1 + i c gamma5)^{-1} = (1 - i c gamma5) / (1 + c^2)
void mdiag_inv_site(double c, const cplx* v, cplx* out) {
    const double d = 1.0 + c * c;
    for (int al = 0; al < 4; ++al)
        for (int a = 0; a < 3; ++a)
            out[3 * al + a] = ((E_ - I_ * (c * GAMMA5[al])) * v[3 * al + a]) / d;
}

Field full_field(const cplx* psi) {
    return [psi](long s, cplx* out) { std::memcpy(out, psi + 12 * s, 12 * sizeof(cplx)); };
}

// A half field living on sites of parity p; reading a site of the other
// parity is a logic error and returns NaN so that a test would catch it.
Field half_field(const Lattice& L, const cplx* half, int p) {
    const Lattice* Lp = &L;
    return [Lp, half, p](long s, cplx* out) {
        int x[4];
        coords(*Lp, s, x);
        if (parity_of(x) != p) {
            for (int i = 0; i < 12; ++i) out[i] = cplx(NAN, NAN);
            return;
        }
        std::memcpy(out, half + 12 * (s / 2), 12 * sizeof(cplx));
    };
}

// out_p[e] = -kappa * bracket(x_e) on all sites of parity p  (D_eo for p = 0).
void dslash_half(const Lattice& L, const cplx* U, const cplx* in, cplx* out, int p,
                 double kappa, double s) {
    Field f = half_field(L, in, 1 - p);
    const long half = L.V / 2;
#pragma omp parallel for schedule(static)
    for (long e = 0; e < half; ++e) {
        int x[4];
        coords(L, lex_of_eo(L, e, p), x);
        cplx acc[12];
        hop_site(L, U, f, x, s, acc);
        for (int i = 0; i < 12; ++i) out[12 * e + i] = -kappa * acc[i];
    }
}

// Mhat(mu)      = M_ee - D_eo M_oo^{-1} D_oe               (dagger = 0, G3)
// Mhat(mu)^dag  = M_ee^dag - D_oe^dag (M_oo^{-1})^dag D_eo^dag   (dagger = 1)
// where X^dag of a hopping block is the adjoint stencil (s = -1) and the
// adjoint of the diagonal is c -> -c.  Acts on even half fields.
void mhat(const Lattice& L, const cplx* U, const cplx* in, cplx* out, double kappa, double mu,
          int dagger) {
    const long half = L.V / 2;
    const double s = dagger ? -1.0 : 1.0;
    const double c = (dagger ? -1.0 : 1.0) * 2.0 * kappa * mu;
    std::vector<cplx> t(12 * half), u(12 * half);
    dslash_half(L, U, in, t.data(), 1, kappa, s);  // odd <- even
    for (long e = 0; e < half; ++e) mdiag_inv_site(c, &t[12 * e], &u[12 * e]);
    dslash_half(L, U, u.data(), t.data(), 0, kappa, s);  // even <- odd
    for (long e = 0; e < half; ++e) {
        cplx d[12];
        mdiag_site(c, in + 12 * e, d);
        for (int i = 0; i < 12; ++i) out[12 * e + i] = d[i] - t[12 * e + i];
    }
}

long double norm2(const cplx* v, long n) {
    long double s = 0.0L;
    for (long i = 0; i < n; ++i)
        s += (long double)v[i].real() * v[i].real() + (long double)v[i].imag() * v[i].imag();
    return s;
}

// Re <a, b> = Re sum conj(a_i) b_i
long double re_dot(const cplx* a, const cplx* b, long n) {
    long double s = 0.0L;
    for (long i = 0; i < n; ++i)
        s += (long double)a[i].real() * b[i].real() + (long double)a[i].imag() * b[i].imag();
    return s;
}

void apply_A(const Lattice& L, const cplx* U, const cplx* in, cplx* out, cplx* tmp, double kappa,
             double mu) {
    mhat(L, U, in, tmp, kappa, mu, 0);
    mhat(L, U, tmp, out, kappa, mu, 1);
}

}  // namespace

extern "C" {

// gamma_mu for which = 0..3, gamma5 for which = 4; out = 16 complex, row-major.
void orc_gamma(int which, double* out) {
    for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b) {
            cplx g = (which < 4) ? GAMMA[which][a][b] : ((a == b) ? cplx(GAMMA5[a], 0) : O_);
            out[2 * (4 * a + b)] = g.real();
            out[2 * (4 * a + b) + 1] = g.imag();
        }
}

// Full operator, eq. 6 with reading G1:  out = (1 + 2 i kappa mu gamma5) psi - kappa * bracket.
// dagger = 1 gives the true adjoint M(mu)^dag (adjoint stencil, c -> -c).
void orc_m_full(const int* dims, const double* bc_phase, const double* U_, const double* in_,
                double* out_, double kappa, double mu, int dagger) {
    Lattice L = make_lattice(dims, bc_phase);
    const cplx* U = (const cplx*)U_;
    const cplx* in = (const cplx*)in_;
    cplx* out = (cplx*)out_;
    Field f = full_field(in);
    const double s = dagger ? -1.0 : 1.0;
    const double c = s * 2.0 * kappa * mu;
#pragma omp parallel for schedule(static)
    for (long sx = 0; sx < L.V; ++sx) {
        int x[4];
        coords(L, sx, x);
        cplx acc[12], d[12];
        hop_site(L, U, f, x, s, acc);
        mdiag_site(c, in + 12 * sx, d);
        for (int i = 0; i < 12; ++i) out[12 * sx + i] = d[i] - kappa * acc[i];
    }
}

// Hopping block: out (parity p half field) = -kappa * bracket applied to `in`
// (parity 1-p half field).  p = 0 is D_eo, p = 1 is D_oe.  adjoint = 1 uses
// the adjoint stencil, i.e. computes (D_{(1-p) p})^dag.
void orc_dslash_eo(const int* dims, const double* bc_phase, const double* U, const double* in,
                   double* out, int parity, double kappa, int adjoint) {
    Lattice L = make_lattice(dims, bc_phase);
    dslash_half(L, (const cplx*)U, (const cplx*)in, (cplx*)out, parity, kappa,
                adjoint ? -1.0 : 1.0);
}

// Same block, but only at the listed output sites (eo indices e of parity p):
// out[k] for k < n_sites.  Used to spot-check full-size lattices site by site.
void orc_dslash_eo_sites(const int* dims, const double* bc_phase, const double* U, const double* in,
                         const long* sites, long n_sites, double* out_, int parity, double kappa,
                         int adjoint) {
    Lattice L = make_lattice(dims, bc_phase);
    Field f = half_field(L, (const cplx*)in, 1 - parity);
    cplx* out = (cplx*)out_;
    for (long k = 0; k < n_sites; ++k) {
        int x[4];
        coords(L, lex_of_eo(L, sites[k], parity), x);
        cplx acc[12];
        hop_site(L, (const cplx*)U, f, x, adjoint ? -1.0 : 1.0, acc);
        for (int i = 0; i < 12; ++i) out[12 * k + i] = -kappa * acc[i];
    }
}

// Even-odd preconditioned operator on even half fields (G3, G11).
void orc_mhat(const int* dims, const double* bc_phase, const double* U, const double* in,
              double* out, double kappa, double mu, int dagger) {
    Lattice L = make_lattice(dims, bc_phase);
    mhat(L, (const cplx*)U, (const cplx*)in, (cplx*)out, kappa, mu, dagger);
}

// Mhat (or its adjoint) at the listed even output sites only, evaluated
// locally: the intermediate odd field u = M_oo^{-1} D_oe in is computed on
// demand at the 8 neighbours of each listed site.
void orc_mhat_sites(const int* dims, const double* bc_phase, const double* U_, const double* in_,
                    const long* sites, long n_sites, double* out_, double kappa, double mu,
                    int dagger) {
    Lattice L = make_lattice(dims, bc_phase);
    const cplx* U = (const cplx*)U_;
    const cplx* in = (const cplx*)in_;
    cplx* out = (cplx*)out_;
    const double s = dagger ? -1.0 : 1.0;
    const double c = s * 2.0 * kappa * mu;
    Field fin = half_field(L, in, 0);
    Field u = [&](long sy, cplx* o) {  // u(y) at an odd site y
        int y[4];
        coords(L, sy, y);
        cplx acc[12], t[12];
        hop_site(L, U, fin, y, s, acc);
        for (int i = 0; i < 12; ++i) t[i] = -kappa * acc[i];
        mdiag_inv_site(c, t, o);
    };
    for (long k = 0; k < n_sites; ++k) {
        int x[4];
        coords(L, lex_of_eo(L, sites[k], 0), x);
        cplx acc[12], d[12];
        hop_site(L, U, u, x, s, acc);
        mdiag_site(c, in + 12 * sites[k], d);
        for (int i = 0; i < 12; ++i) out[12 * k + i] = d[i] - (-kappa * acc[i]);
    }
}

// Textbook Hestenes-Stiefel CG on A = Mhat^dag Mhat, even half fields, x0 = 0
// (G10): r = p = b, rho = |r|^2; loop: q = A p; alpha = rho / Re<p,q>;
// x += alpha p; r -= alpha q; rho' = |r|^2; stop if rho' <= tol^2 |b|^2;
// p = r + (rho'/rho) p.  Returns 0 converged, 1 not converged after maxit
// iterations (x = last iterate), -5 breakdown (Re<p,q> <= 0 or not finite).
int orc_cg_mdagm(const int* dims, const double* bc_phase, const double* U_, const double* b_,
                 double* x_, double kappa, double mu, double tol, int maxit, int* iters,
                 double* rel_resid_recursive, double* rel_resid_true) {
    Lattice L = make_lattice(dims, bc_phase);
    const cplx* U = (const cplx*)U_;
    const cplx* b = (const cplx*)b_;
    cplx* x = (cplx*)x_;
    const long n = 12 * (L.V / 2);
    std::vector<cplx> r(b, b + n), p(b, b + n), q(n), tmp(n);
    for (long i = 0; i < n; ++i) x[i] = O_;
    const long double bb = norm2(b, n);
    long double rho = bb;
    int it = 0, status = 1;
    if (bb == 0.0L) {
        status = 0;
    } else {
        while (it < maxit) {
            apply_A(L, U, p.data(), q.data(), tmp.data(), kappa, mu);
            const long double pq = re_dot(p.data(), q.data(), n);
            if (!(pq > 0.0L) || !std::isfinite((double)pq)) { status = -5; break; }
            const double alpha = (double)(rho / pq);
            for (long i = 0; i < n; ++i) x[i] += alpha * p[i];
            for (long i = 0; i < n; ++i) r[i] -= alpha * q[i];
            const long double rho1 = norm2(r.data(), n);
            ++it;
            if (rho1 <= (long double)tol * tol * bb) { rho = rho1; status = 0; break; }
            const double beta = (double)(rho1 / rho);
            for (long i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
            rho = rho1;
        }
    }
    if (iters) *iters = it;
    if (rel_resid_recursive) *rel_resid_recursive = bb > 0 ? (double)sqrtl(rho / bb) : 0.0;
    if (rel_resid_true) {
        apply_A(L, U, x, q.data(), tmp.data(), kappa, mu);
        for (long i = 0; i < n; ++i) q[i] = b[i] - q[i];
        *rel_resid_true = bb > 0 ? (double)sqrtl(norm2(q.data(), n) / bb) : 0.0;
    }
    return status;
}

// BiCGStab (van der Vorst, SIAM J. Sci. Stat. Comput. 13 (1992) 631) on Mhat x = b, even half
// fields, x0 = 0 -- the second solver the paper names ("The most common solvers used are CG and
// BiCGStab").  The paper gives no formulae; reading G15 of DESIGN.md: the
// textbook recurrence with shadow residual rhat = r0 = b and p0 = r0, complex inner product
// <a,b> = sum conj(a_i) b_i, one iteration = two applications of Mhat:
//   rho = <rhat, r>;  loop: v = Mhat p; sigma = <rhat, v>; alpha = rho / sigma; s = r - alpha v;
//   t = Mhat s; omega = <t,s>/<t,t> (0 if t = 0); x += alpha p + omega s; r = s - omega t;
//   stop if |r| <= tol |b|; rho' = <rhat, r>; beta = (rho'/rho)(alpha/omega);
//   p = r + beta (p - omega v); rho = rho'.
// Returns 0 converged, 1 not converged after maxit iterations (x = last iterate), -5 breakdown
// (sigma, rho' or omega zero or not finite).
int orc_bicgstab_mhat(const int* dims, const double* bc_phase, const double* U_, const double* b_,
                      double* x_, double kappa, double mu, double tol, int maxit, int* iters,
                      double* rel_resid_recursive, double* rel_resid_true) {
    Lattice L = make_lattice(dims, bc_phase);
    const cplx* U = (const cplx*)U_;
    const cplx* b = (const cplx*)b_;
    cplx* x = (cplx*)x_;
    const long n = 12 * (L.V / 2);
    typedef std::complex<long double> lcplx;
    auto cdot = [n](const cplx* a, const cplx* c) {  // <a, c> = sum conj(a_i) c_i
        lcplx s(0.0L, 0.0L);
        for (long i = 0; i < n; ++i) s += std::conj(lcplx(a[i])) * lcplx(c[i]);
        return s;
    };
    auto bad = [](cplx z) { return z == O_ || !std::isfinite(z.real()) || !std::isfinite(z.imag()); };
    std::vector<cplx> r(b, b + n), p(b, b + n), v(n), s(n), t(n);
    const cplx* rhat = b;
    for (long i = 0; i < n; ++i) x[i] = O_;
    const long double bb = norm2(b, n);
    long double rr = bb;
    int it = 0, status = 1;
    if (bb == 0.0L) {
        status = 0;
    } else {
        cplx rho = (cplx)cdot(rhat, r.data());
        while (it < maxit) {
            mhat(L, U, p.data(), v.data(), kappa, mu, 0);
            const cplx sigma = (cplx)cdot(rhat, v.data());
            if (bad(sigma)) { status = -5; break; }
            const cplx alpha = rho / sigma;
            for (long i = 0; i < n; ++i) s[i] = r[i] - alpha * v[i];
            mhat(L, U, s.data(), t.data(), kappa, mu, 0);
            const long double tt = norm2(t.data(), n);
            const cplx omega = tt > 0.0L ? (cplx)(cdot(t.data(), s.data()) / tt) : O_;
            for (long i = 0; i < n; ++i) x[i] += alpha * p[i] + omega * s[i];
            for (long i = 0; i < n; ++i) r[i] = s[i] - omega * t[i];
            rr = norm2(r.data(), n);
            ++it;
            if (rr <= (long double)tol * tol * bb) { status = 0; break; }
            const cplx rho1 = (cplx)cdot(rhat, r.data());
            if (bad(rho1) || bad(omega)) { status = -5; break; }
            const cplx beta = (rho1 / rho) * (alpha / omega);
            for (long i = 0; i < n; ++i) p[i] = r[i] + beta * (p[i] - omega * v[i]);
            rho = rho1;
        }
    }
    if (iters) *iters = it;
    if (rel_resid_recursive) *rel_resid_recursive = bb > 0 ? (double)sqrtl(rr / bb) : 0.0;
    if (rel_resid_true) {
        mhat(L, U, x, t.data(), kappa, mu, 0);
        for (long i = 0; i < n; ++i) t[i] = b[i] - t[i];
        *rel_resid_true = bb > 0 ? (double)sqrtl(norm2(t.data(), n) / bb) : 0.0;
    }
    return status;
}

// A = Mhat^dag Mhat applied once (the operator CG inverts).
void orc_mdagm(const int* dims, const double* bc_phase, const double* U, const double* in,
               double* out, double kappa, double mu) {
    Lattice L = make_lattice(dims, bc_phase);
    std::vector<cplx> tmp(12 * (L.V / 2));
    apply_A(L, (const cplx*)U, (const cplx*)in, (cplx*)out, tmp.data(), kappa, mu);
}

// ---------------------------------------------------------------------------
// Fermion force (eq. 9-10; Table 2 row F_fermion, PAPER.md:236;
// Table 3 "P, F: (N_C^2 - 1) x N_D" reals per site).
//
// The paper states F = -dS/dU (eq. 9), that F_mu(x) is a real (N_C^2 - 1)-vector, that it
// follows from d(D^-1) = -D^-1 (dD) D^-1 and that only the hopping part of the matrix
// contributes; it prints no formula.  Reading G16 of DESIGN.md:
//   * components are taken along T^a = lambda^a / 2 (Gell-Mann matrices, standard order),
//     with the link varied from the left:  U_mu(x) -> exp(i w T^a) U_mu(x),
//     F^a_mu(x) = - dS/dw at w = 0;
//   * for two spinor fields X, Y on the whole lattice the "outer product" force is
//     F^a_mu(x) = 2 Re d/dw [ Y^dag D(w) X ]
//               = 2 kappa Im [ Y(x)^dag T^a a(x) - b(x)^dag T^a X(x) ],
//     a(x) = eta+_mu(x) (1 - gamma_mu) U_mu(x) X(x+mu),  b(x) = eta+_mu(x) (1 + gamma_mu) U_mu(x) Y(x+mu),
//     which is what dS = -2 Re (Y^dag dD X) gives for S = phi^dag (M^dag M)^-1 phi with
//     X = (M^dag M)^-1 phi, Y = M X (the minus of F = -dS/dU cancels the minus of d(A^-1));
//   * for the even-odd action S = phi_e^dag (Mhat^dag Mhat)^-1 phi_e the same formula holds
//     with X_e = (Mhat^dag Mhat)^-1 phi, Y_e = Mhat X_e, X_o = -M_oo^-1 D_oe X_e,
//     Y_o = -(M_oo^-1)^dag (D_eo)^dag Y_e, since d Mhat = -dD_eo M_oo^-1 D_oe - D_eo M_oo^-1 dD_oe.
// Pinned in tests/test_oracle_pins.py (P10) by central differences of S computed from
// dense matrices in numpy, and by gauge covariance.
// ---------------------------------------------------------------------------

namespace {

// Gell-Mann matrices lambda^1..lambda^8, row-major.
void gell_mann(int a, cplx* l) {
    for (int i = 0; i < 9; ++i) l[i] = O_;
    const double s3 = 1.0 / std::sqrt(3.0);
    switch (a) {
        case 0: l[1] = E_; l[3] = E_; break;
        case 1: l[1] = -I_; l[3] = I_; break;
        case 2: l[0] = E_; l[4] = -E_; break;
        case 3: l[2] = E_; l[6] = E_; break;
        case 4: l[2] = -I_; l[6] = I_; break;
        case 5: l[5] = E_; l[7] = E_; break;
        case 6: l[5] = -I_; l[7] = I_; break;
        case 7: l[0] = s3; l[4] = s3; l[8] = -2.0 * s3; break;
    }
}

// u^dag T^a v for two spinors (sum over Dirac and colour), T^a = lambda^a / 2
cplx sandwich(const cplx* u, int a, const cplx* v) {
    cplx lam[9];
    gell_mann(a, lam);
    cplx s = O_;
    for (int al = 0; al < 4; ++al)
        for (int c = 0; c < 3; ++c)
            for (int d = 0; d < 3; ++d) s += std::conj(u[3 * al + c]) * (0.5 * lam[3 * c + d]) * v[3 * al + d];
    return s;
}

// F^a_mu(x), a = 0..7, for the link U_mu(x): the formula of reading G16 written out.
void force_link(const Lattice& L, const cplx* U, const cplx* X, const cplx* Y, const int* x, int mu,
                double kappa, double* F8) {
    const long sx = lex(L, x);
    int y[4] = {x[0], x[1], x[2], x[3]};
    y[mu] = (x[mu] + 1) % L.N[mu];
    const long sy = lex(L, y);
    const cplx eta = (x[mu] == L.N[mu] - 1) ? L.phase[mu] : E_;
    cplx t[12], a[12], b[12];
    su3_mul(U + (sx * 4 + mu) * 9, X + 12 * sy, t);
    one_plus_sgamma(mu, -1.0, t, a);
    su3_mul(U + (sx * 4 + mu) * 9, Y + 12 * sy, t);
    one_plus_sgamma(mu, +1.0, t, b);
    for (int i = 0; i < 12; ++i) { a[i] *= eta; b[i] *= eta; }
    for (int g = 0; g < 8; ++g)
        F8[g] = 2.0 * kappa * (sandwich(Y + 12 * sx, g, a) - sandwich(b, g, X + 12 * sx)).imag();
}

}  // namespace

// Outer-product force for two full-lattice spinor fields (canonical layouts):
// F[lex(x)][mu][a], a = 0..7 real.
void orc_fermion_force(const int* dims, const double* bc_phase, const double* U_, const double* X_,
                       const double* Y_, double kappa, double* F) {
    Lattice L = make_lattice(dims, bc_phase);
#pragma omp parallel for schedule(static)
    for (long sx = 0; sx < L.V; ++sx) {
        int x[4];
        coords(L, sx, x);
        for (int mu = 0; mu < 4; ++mu)
            force_link(L, (const cplx*)U_, (const cplx*)X_, (const cplx*)Y_, x, mu, kappa, F + (sx * 4 + mu) * 8);
    }
}

// The same at the listed links only: link k is (lex site sites[k], direction mus[k]).
void orc_fermion_force_links(const int* dims, const double* bc_phase, const double* U_, const double* X_,
                             const double* Y_, const long* sites, const int* mus, long n_links, double kappa,
                             double* F) {
    Lattice L = make_lattice(dims, bc_phase);
    for (long k = 0; k < n_links; ++k) {
        int x[4];
        coords(L, sites[k], x);
        force_link(L, (const cplx*)U_, (const cplx*)X_, (const cplx*)Y_, x, mus[k], kappa, F + 8 * k);
    }
}

// Fields of the even-odd force from a solution X_e:  Y_e = Mhat X_e, X_o = -M_oo^-1 D_oe X_e,
// Y_o = -(M_oo^-1)^dag (D_eo)^dag Y_e, returned as full-lattice fields X, Y (canonical).
void orc_force_fields(const int* dims, const double* bc_phase, const double* U_, const double* Xe_,
                      double kappa, double mu, double* X_, double* Y_) {
    Lattice L = make_lattice(dims, bc_phase);
    const cplx* U = (const cplx*)U_;
    const cplx* Xe = (const cplx*)Xe_;
    cplx* X = (cplx*)X_;
    cplx* Y = (cplx*)Y_;
    const long half = L.V / 2;
    const double c = 2.0 * kappa * mu;
    std::vector<cplx> Ye(12 * half), t(12 * half), Xo(12 * half), Yo(12 * half);
    mhat(L, U, Xe, Ye.data(), kappa, mu, 0);
    dslash_half(L, U, Xe, t.data(), 1, kappa, +1.0);            // D_oe X_e
    for (long e = 0; e < half; ++e) {
        mdiag_inv_site(c, &t[12 * e], &Xo[12 * e]);
        for (int i = 0; i < 12; ++i) Xo[12 * e + i] = -Xo[12 * e + i];
    }
    dslash_half(L, U, Ye.data(), t.data(), 1, kappa, -1.0);     // (D_eo)^dag Y_e: adjoint stencil, odd sites
    for (long e = 0; e < half; ++e) {
        mdiag_inv_site(-c, &t[12 * e], &Yo[12 * e]);            // (M_oo^-1)^dag
        for (int i = 0; i < 12; ++i) Yo[12 * e + i] = -Yo[12 * e + i];
    }
    for (long e = 0; e < half; ++e) {
        const long se = lex_of_eo(L, e, 0), so = lex_of_eo(L, e, 1);
        for (int i = 0; i < 12; ++i) {
            X[12 * se + i] = Xe[12 * e + i]; Y[12 * se + i] = Ye[12 * e + i];
            X[12 * so + i] = Xo[12 * e + i]; Y[12 * so + i] = Yo[12 * e + i];
        }
    }
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// Thread count of the OpenMP loops over independent output sites (no arithmetic changes with it): the
// timed baseline is reported once single-threaded and once on all cores.
// n <= 0 restores the default; returns the count now in force.
int orc_set_num_threads(int n) {
#ifdef _OPENMP
    static const int dflt = omp_get_max_threads();
    omp_set_num_threads(n > 0 ? n : dflt);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}

}  // extern "C"
