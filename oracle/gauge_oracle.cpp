// gauge_oracle.cpp -- TEST INFRASTRUCTURE ONLY.
//
// A plain, slow CPU statement of the paper's second workload, the pure-gauge heatbath and
// overrelaxation update (Fig. 2; Table 2 rows "heatbath" / "overrelax",
// PAPER.md:237-238).  Same rules as lqcd_oracle.cpp: only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline leg may call this; it shares no code,
// header, table or helper with the CUDA path; std::complex<double>, -ffp-contract=off.
//
// What the paper fixes: the gauge action (eq. 5; "the unimproved gauge action
// is regained setting c_1 to zero"), and Fig. 2:
//     L(0) = U;  for i < m = #subgroups:  W = L(i) * Staple;  w = project(W, i);
//     v = update(w);  V = extend(v, i);  L(i) = L(i-1) * V;   U = L(m)
// with "update" the exact SU(2) heatbath [16-18] or an overrelaxation step [19], m = 3 subgroups
// for SU(3), and random numbers needed "only in the first update" (the heatbath).
// Everything else is a reading (G17-G21):
//   G17 action: Wilson plaquette action, S = beta sum_x sum_{mu<nu} (1 - Re tr P_mu_nu(x) / 3)
//       (eq. 5 with c_1 = 0; the paper's 2880 B per link for both kernels, is
//       exactly 1 link + 6 staples x 3 links + 1 store, i.e. plaquette staples only).  The
//       gauge field is periodic (the boundary phases of lqcd_init belong to the fermions).
//   G18 the product order that is consistent with W = L * Staple is LEFT multiplication,
//       L(i) = V * L(i-1): tr(V L A) = tr(V W).  (Fig. 2 is a "sketch"; with L * V the matrix
//       to project would be Staple * L.)
//   G19 subgroups in the order (0,1), (1,2), (0,2); SU(2) element a0 + i (a1 s1 + a2 s2 + a3 s3)
//       = [[a0 + i a3, a2 + i a1], [-a2 + i a1, a0 - i a3]]; project(W) takes
//       a0 = Re(W_pp + W_qq)/2, a1 = Im(W_pq + W_qp)/2, a2 = Re(W_pq - W_qp)/2,
//       a3 = Im(W_pp - W_qq)/2, k = |a|, w = a / k.
//   G20 heatbath = Kennedy-Pendleton [18]: the new g = v w has density sqrt(1 - g0^2)
//       exp(lambda g0), lambda = 2 beta k / 3; draw r1..r4 in (0,1], delta = -(ln r1 +
//       cos^2(2 pi r2) ln r3) / lambda, accept if r4^2 <= 1 - delta/2, g0 = 1 - delta; after
//       MAXTRY = 32 rejections the subgroup is left unchanged (v = 1), which keeps detailed
//       balance because the failure probability depends on the staple only.  Direction uniform
//       on the sphere: cos(theta) = 2 r5 - 1, phi = 2 pi r6.  v = g w^dag.
//       overrelax: v = (w^dag)^2, so that v w = w^dag has the same trace as w (action unchanged).
//       k = 0 (no preferred direction): the subgroup is skipped.
//   G21 random numbers: the counter-based generator of the input recipe,
//       u = uniform(seed, stream = tag, counter), counter = (((4 lex(x) + mu) * 3 + i) * 33 +
//       attempt) * 4 + j; the two direction draws use attempt = 32, j = 0, 1.  The CUDA path
//       implements the same generator on its own.
//   Update order of a sweep: mu = 0..3, inside it parity 0 then 1; all links of one (mu, parity)
//       are independent (their staples hold no link of that set).
//
// Pins (tests/test_gauge_oracle_pins.py, -m "not gpu"): plaquette and action against an
// independent numpy build with np.roll, the staple through the exact identity
// S[U'] - S[U] = -(beta/3) Re tr((U' - U) A) (P11); overrelaxation keeps the action, keeps
// SU(3), and reduces to the textbook SU(2) formula U' = V^dag U^dag V^dag on a field embedded in
// one subgroup (P12); the Kennedy-Pendleton sampler against the closed form <g0> =
// I_2(lambda) / I_1(lambda) and the strong-coupling plaquette <P> = beta/18 + beta^2/216 (P13).

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

typedef std::complex<double> cplx;
const cplx I_(0.0, 1.0);

struct Lat {
    int N[4];
    long V;
};

Lat make_lat(const int* dims) {
    Lat L;
    L.V = 1;
    for (int m = 0; m < 4; ++m) { L.N[m] = dims[m]; L.V *= dims[m]; }
    return L;
}
long lex(const Lat& L, const int* x) {
    return x[0] + (long)L.N[0] * (x[1] + (long)L.N[1] * (x[2] + (long)L.N[2] * x[3]));
}
void coords(const Lat& L, long s, int* x) {
    x[0] = (int)(s % L.N[0]); s /= L.N[0];
    x[1] = (int)(s % L.N[1]); s /= L.N[1];
    x[2] = (int)(s % L.N[2]); s /= L.N[2];
    x[3] = (int)s;
}
// lex index of x + d1 * e_m1 + d2 * e_m2 (periodic)
long shifted(const Lat& L, const int* x, int m1, int d1, int m2 = 0, int d2 = 0) {
    int y[4] = {x[0], x[1], x[2], x[3]};
    y[m1] = (y[m1] + d1 + L.N[m1]) % L.N[m1];
    y[m2] = (y[m2] + d2 + L.N[m2]) % L.N[m2];
    return lex(L, y);
}

// 3x3 complex matrices, row-major
void mm(const cplx* a, const cplx* b, cplx* c) {           // c = a b
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            cplx s = 0.0;
            for (int k = 0; k < 3; ++k) s += a[3 * i + k] * b[3 * k + j];
            c[3 * i + j] = s;
        }
}
void dag(const cplx* a, cplx* c) {                          // c = a^dag
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c[3 * i + j] = std::conj(a[3 * j + i]);
}
const cplx* link(const cplx* U, long s, int mu) { return U + (s * 4 + mu) * 9; }

// Staple sum of the link U_mu(x): Re tr(U_mu(x) A) = sum of Re tr over the 6 plaquettes that
// contain the link (the "staple P~_mu_nu(x): the plaquette product of links without U_mu(x)",
// PAPER.md:110, fig. 1):
//   A = sum_{nu != mu} [ U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
//                      + U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu) ]
void staple(const Lat& L, const cplx* U, const int* x, int mu, cplx* A) {
    for (int i = 0; i < 9; ++i) A[i] = 0.0;
    const long sx = lex(L, x);
    cplx d1[9], d2[9], t[9], p[9];
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        // forward: x -> x+mu -> x+mu+nu -> x+nu -> x
        dag(link(U, shifted(L, x, nu, +1), mu), d1);
        dag(link(U, sx, nu), d2);
        mm(link(U, shifted(L, x, mu, +1), nu), d1, t);
        mm(t, d2, p);
        for (int i = 0; i < 9; ++i) A[i] += p[i];
        // backward: x -> x+mu -> x+mu-nu -> x-nu -> x
        dag(link(U, shifted(L, x, mu, +1, nu, -1), nu), d1);
        dag(link(U, shifted(L, x, nu, -1), mu), d2);
        mm(d1, d2, t);
        mm(t, link(U, shifted(L, x, nu, -1), nu), p);
        for (int i = 0; i < 9; ++i) A[i] += p[i];
    }
}

// Counter-based uniform in (0,1] of the input recipe, restated:
// bits = splitmix64_mix(seed * GOLD + stream * 2^40 + counter); u = (top 53 bits + 1) / 2^53.
double uniform01(uint64_t seed, uint64_t stream, uint64_t counter) {
    uint64_t z = seed * 0x9E3779B97F4A7C15ULL + (stream << 40) + counter;
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return ((double)(z >> 11) + 1.0) * (1.0 / 9007199254740992.0);
}

const int MAXTRY = 32;
const int SUB_P[3] = {0, 1, 0};
const int SUB_Q[3] = {1, 2, 2};

// SU(2) elements as 2x2 complex matrices, [[a0 + i a3, a2 + i a1], [-a2 + i a1, a0 - i a3]] (G19)
void su2_matrix(const double* a, cplx* m) {
    m[0] = cplx(a[0], a[3]);  m[1] = cplx(a[2], a[1]);
    m[2] = cplx(-a[2], a[1]); m[3] = cplx(a[0], -a[3]);
}
void mm2(const cplx* a, const cplx* b, cplx* c) {
    c[0] = a[0] * b[0] + a[1] * b[2]; c[1] = a[0] * b[1] + a[1] * b[3];
    c[2] = a[2] * b[0] + a[3] * b[2]; c[3] = a[2] * b[1] + a[3] * b[3];
}
void dag2(const cplx* a, cplx* c) {
    c[0] = std::conj(a[0]); c[1] = std::conj(a[2]);
    c[2] = std::conj(a[1]); c[3] = std::conj(a[3]);
}

// Kennedy-Pendleton (G20): g with density sqrt(1 - g0^2) exp(lambda g0) dg0 x uniform direction.
// `base` is the counter of (attempt 0, j = 0).  Returns the number of attempts used (1..MAXTRY),
// or 0 if all were rejected (g is then not set).
int kp_sample(double lambda, uint64_t seed, uint64_t tag, uint64_t base, double* g) {
    const double two_pi = 6.283185307179586476925286766559;
    for (int attempt = 0; attempt < MAXTRY; ++attempt) {
        const uint64_t c = base + 4 * (uint64_t)attempt;
        const double r1 = uniform01(seed, tag, c), r2 = uniform01(seed, tag, c + 1);
        const double r3 = uniform01(seed, tag, c + 2), r4 = uniform01(seed, tag, c + 3);
        const double cs = std::cos(two_pi * r2);
        const double delta = -(std::log(r1) + cs * cs * std::log(r3)) / lambda;
        if (r4 * r4 <= 1.0 - 0.5 * delta) {
            const uint64_t cd = base + 4 * (uint64_t)MAXTRY;
            const double r5 = uniform01(seed, tag, cd), r6 = uniform01(seed, tag, cd + 1);
            const double g0 = 1.0 - delta;
            const double rad = std::sqrt(1.0 - g0 * g0);
            const double ct = 2.0 * r5 - 1.0;
            const double st = std::sqrt(1.0 - ct * ct);
            const double phi = two_pi * r6;
            g[0] = g0;
            g[1] = rad * st * std::cos(phi);
            g[2] = rad * st * std::sin(phi);
            g[3] = rad * ct;
            return attempt + 1;
        }
    }
    return 0;
}

// Fig. 2 for one link: Lk (in: U_mu(x), out: the updated link), A its staple sum.
// mode 0 = heatbath, 1 = overrelax; `subgroups` is a bit mask of the steps i = 0, 1, 2 to do
// (7 = the algorithm; single steps exist for the pins).
void update_link(cplx* Lk, const cplx* A, int mode, int subgroups, double beta, uint64_t seed,
                 uint64_t tag, uint64_t link_id) {
    for (int i = 0; i < 3; ++i) {
        if (!((subgroups >> i) & 1)) continue;
        const int p = SUB_P[i], q = SUB_Q[i];
        cplx W[9];
        mm(Lk, A, W);                                            // W = L(i) * Staple
        double a[4];                                             // w = project(W, i)   (G19)
        a[0] = 0.5 * (W[3 * p + p].real() + W[3 * q + q].real());
        a[1] = 0.5 * (W[3 * p + q].imag() + W[3 * q + p].imag());
        a[2] = 0.5 * (W[3 * p + q].real() - W[3 * q + p].real());
        a[3] = 0.5 * (W[3 * p + p].imag() - W[3 * q + q].imag());
        const double k = std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2] + a[3] * a[3]);
        if (!(k > 0.0)) continue;
        for (int j = 0; j < 4; ++j) a[j] /= k;
        cplx w[4], wd[4], v[4];
        su2_matrix(a, w);
        dag2(w, wd);
        if (mode == 0) {                                         // v = update(w): heatbath
            double g[4];
            const uint64_t base = ((link_id * 3 + (uint64_t)i) * (uint64_t)(MAXTRY + 1)) * 4;
            if (kp_sample(2.0 * beta * k / 3.0, seed, tag, base, g) == 0) continue;
            cplx gm[4];
            su2_matrix(g, gm);
            mm2(gm, wd, v);                                      // v w = g
        } else {                                                 // overrelax: v w = w^dag
            mm2(wd, wd, v);
        }
        cplx Vx[9], Ln[9];                                       // V = extend(v, i)
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c) Vx[3 * r + c] = (r == c) ? 1.0 : 0.0;
        Vx[3 * p + p] = v[0]; Vx[3 * p + q] = v[1];
        Vx[3 * q + p] = v[2]; Vx[3 * q + q] = v[3];
        mm(Vx, Lk, Ln);                                          // L(i) = V * L(i-1)   (G18)
        std::memcpy(Lk, Ln, sizeof(Ln));
    }
}

}  // namespace

extern "C" {

// Average plaquette (1/3) Re tr P_mu_nu(x) over the 6 V plaquettes (eq. 5 with c_1 = 0),
// P_mu_nu(x) = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag.  Sum in long double.
double orc_plaquette(const int* dims, const double* U_) {
    Lat L = make_lat(dims);
    const cplx* U = (const cplx*)U_;
    long double sum = 0.0L;
    for (long s = 0; s < L.V; ++s) {
        int x[4];
        coords(L, s, x);
        for (int mu = 0; mu < 4; ++mu)
            for (int nu = mu + 1; nu < 4; ++nu) {
                cplx d1[9], d2[9], t1[9], t2[9], P[9];
                dag(link(U, shifted(L, x, nu, +1), mu), d1);
                dag(link(U, s, nu), d2);
                mm(link(U, s, mu), link(U, shifted(L, x, mu, +1), nu), t1);
                mm(t1, d1, t2);
                mm(t2, d2, P);
                sum += (long double)((P[0] + P[4] + P[8]).real() / 3.0);
            }
    }
    return (double)(sum / (long double)(6 * L.V));
}

// Staple sum A of the link (lex site, mu): 9 complex, row-major.
void orc_staple(const int* dims, const double* U_, long site, int mu, double* A_) {
    Lat L = make_lat(dims);
    int x[4];
    coords(L, site, x);
    staple(L, (const cplx*)U_, x, mu, (cplx*)A_);
}

// Fig. 2 for the listed links of the field U, each from the SAME input field (nothing is
// written back): out[k] = the updated U_mus[k](sites[k]).  mode 0 heatbath, 1 overrelax;
// subgroups = 7 for the algorithm.
void orc_update_links(const int* dims, const double* U_, const long* sites, const int* mus,
                      long n_links, int mode, int subgroups, double beta,
                      unsigned long long seed, unsigned long long tag, double* out_) {
    Lat L = make_lat(dims);
    const cplx* U = (const cplx*)U_;
    cplx* out = (cplx*)out_;
    for (long k = 0; k < n_links; ++k) {
        int x[4];
        coords(L, sites[k], x);
        cplx A[9], Lk[9];
        staple(L, U, x, mus[k], A);
        std::memcpy(Lk, link(U, sites[k], mus[k]), sizeof(Lk));
        update_link(Lk, A, mode, subgroups, beta, seed, tag, (uint64_t)(4 * sites[k] + mus[k]));
        std::memcpy(out + 9 * k, Lk, sizeof(Lk));
    }
}

// One sub-sweep in place: every link U_mu(x) with parity(x) = parity.  These links are
// independent (no staple of the set holds a link of the set), so the loop order is immaterial.
void orc_gauge_subsweep(const int* dims, double* U_, int mu, int parity, int mode, double beta,
                        unsigned long long seed, unsigned long long tag) {
    Lat L = make_lat(dims);
    cplx* U = (cplx*)U_;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < L.V; ++s) {
        int x[4];
        coords(L, s, x);
        if (((x[0] + x[1] + x[2] + x[3]) & 1) != parity) continue;
        cplx A[9];
        staple(L, U, x, mu, A);
        update_link(U + (s * 4 + mu) * 9, A, mode, 7, beta, seed, tag, (uint64_t)(4 * s + mu));
    }
}

// One sweep in place: mu = 0..3, parity 0 then 1.
void orc_gauge_sweep(const int* dims, double* U, int mode, double beta, unsigned long long seed,
                     unsigned long long tag) {
    for (int mu = 0; mu < 4; ++mu)
        for (int parity = 0; parity < 2; ++parity)
            orc_gauge_subsweep(dims, U, mu, parity, mode, beta, seed, tag);
}

// The Kennedy-Pendleton sampler alone (for the distribution pin): n samples with counters
// base = 4 * 33 * j, j = 0..n-1; g[4 j ..], attempts[j] (0 = all 32 rejected, g = 0).
void orc_kp_samples(double lambda, unsigned long long seed, unsigned long long tag, long n,
                    double* g, int* attempts) {
    for (long j = 0; j < n; ++j) {
        double q[4] = {0.0, 0.0, 0.0, 0.0};
        attempts[j] = kp_sample(lambda, seed, tag, (uint64_t)j * 4 * (MAXTRY + 1), q);
        for (int c = 0; c < 4; ++c) g[4 * j + c] = q[c];
    }
}

}  // extern "C"
