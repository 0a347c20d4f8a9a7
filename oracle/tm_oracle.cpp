// oracle/tm_oracle.cpp
//
// TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 CPU oracle for the hot path of
// arxiv/paper_1309_2256 (twisted-mass Wilson operator, even-odd preconditioning, CG,
// stochastic loop contraction).  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, load or call this file.  It shares no
// code with the CUDA library (paper_1309_2256_b200/csrc) and neither includes the other.
//
// Everything here is the plain definition written out: full-lattice fields in the canonical
// layout, full 3x3 links, dense 4x4 gamma matrices multiplied out naively -- no spin
// projection trick, no even-odd storage, no link reconstruction, no blocking.
// Parity-restricted operators are the full operator between parity projectors.
//
// Conventions:
//   site = x + X*(y + Y*(z + Z*t)); mu = 0..3 = x,y,z,t; parity = (x+y+z+t)&1, even = 0.
//   gauge U[site][mu][row][col], spinor psi[site][spin][colour], complex fp64 interleaved.
//   Periodic in space; time antiperiodic when `ap` != 0: the hop across t=T-1 <-> 0 carries -1.
//   Dslash (positive hopping sum; "H = 2 kappa D, with D the hopping term", D = -Dslash/2):
//     (Dslash psi)(x) = sum_mu (1-g_mu) s_mu(x) U_mu(x) psi(x+mu) + (1+g_mu) s_mu(x-mu) U_mu(x-mu)^dag psi(x-mu)
//   M(kappa,mu) = 1 + i*2*kappa*mu*g5 - kappa*Dslash   (PAPER.md:162 B^-1 = 1 + i 2 kappa mu a g5; :367 Eq. A1)
//   gamma basis: chiral, g_k = [[0,-i s_k],[i s_k,0]], g_4 = [[0,1],[1,0]], g5 = g1 g2 g3 g4.
//
// Pins: tests/test_oracle_pins.py (free-field closed form, g5-hermiticity, gauge covariance,
// dense brute force on 4^4 built independently in numpy, HPE identity Eq. 16, exact traces).
#include <complex>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

typedef std::complex<double> cd;
static const cd I_(0.0, 1.0);

struct Geom {
    int X, Y, Z, T, ap;
    long V;
    Geom(const int* d, int ap_) : X(d[0]), Y(d[1]), Z(d[2]), T(d[3]), ap(ap_), V((long)d[0] * d[1] * d[2] * d[3]) {}
    long idx(int x, int y, int z, int t) const { return x + (long)X * (y + (long)Y * (z + (long)Z * t)); }
    void coords(long i, int c[4]) const {
        c[0] = (int)(i % X); i /= X;
        c[1] = (int)(i % Y); i /= Y;
        c[2] = (int)(i % Z); i /= Z;
        c[3] = (int)i;
    }
    int len(int mu) const { return mu == 0 ? X : mu == 1 ? Y : mu == 2 ? Z : T; }
    int parity(long i) const { int c[4]; coords(i, c); return (c[0] + c[1] + c[2] + c[3]) & 1; }
};

// ---------------------------------------------------------------------------------------
// gamma matrices, SURVEY.md 8(c-1) item 3 (reading of PAPER.md:369 -- external basis unstated)
// ---------------------------------------------------------------------------------------
static void gamma_mu(int mu, cd g[4][4])
{
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) g[a][b] = 0.0;
    // Pauli matrices
    cd s[3][2][2] = {{{0, 1}, {1, 0}}, {{0, -I_}, {I_, 0}}, {{1, 0}, {0, -1}}};
    if (mu < 3) {
        for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) {
            g[a][2 + b] = -I_ * s[mu][a][b];
            g[2 + a][b] = I_ * s[mu][a][b];
        }
    } else if (mu == 3) {
        g[0][2] = g[1][3] = g[2][0] = g[3][1] = 1.0;
    } else { // gamma5 = g1 g2 g3 g4
        cd p[4][4], q[4][4], t[4][4];
        gamma_mu(0, p);
        for (int k = 1; k < 4; ++k) {
            gamma_mu(k, q);
            for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
                t[a][b] = 0.0;
                for (int c = 0; c < 4; ++c) t[a][b] += p[a][c] * q[c][b];
            }
            std::memcpy(p, t, sizeof(t));
        }
        std::memcpy(g, p, sizeof(p));
    }
}

// Gamma_n = g1^b0 g2^b1 g3^b2 g4^b3, n = b0 + 2 b1 + 4 b2 + 8 b3  (reading 15: "all the possible
// insertions for ultra-local operators"; ordered products, no factors of i)
static void Gamma_n(int n, cd G[4][4])
{
    cd p[4][4], q[4][4], t[4][4];
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) p[a][b] = (a == b) ? 1.0 : 0.0;
    for (int k = 0; k < 4; ++k) {
        if (!((n >> k) & 1)) continue;
        gamma_mu(k, q);
        for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
            t[a][b] = 0.0;
            for (int c = 0; c < 4; ++c) t[a][b] += p[a][c] * q[c][b];
        }
        std::memcpy(p, t, sizeof(t));
    }
    std::memcpy(G, p, sizeof(p));
}

extern "C" void orc_gamma(int mu, double* out) { cd g[4][4]; gamma_mu(mu, g); std::memcpy(out, g, sizeof(g)); }
extern "C" void orc_Gamma(int n, double* out) { cd g[4][4]; Gamma_n(n, g); std::memcpy(out, g, sizeof(g)); }

// ---------------------------------------------------------------------------------------
// hopping term, full lattice.  dagger: Dslash^dag = g5 Dslash g5 (every g_mu -> -g_mu).
// ---------------------------------------------------------------------------------------
static void hop_site(const Geom& G, const cd* U, const cd* in, long i, int dagger, cd out[12])
{
    int c[4];
    G.coords(i, c);
    for (int k = 0; k < 12; ++k) out[k] = 0.0;
    for (int mu = 0; mu < 4; ++mu) {
        cd g[4][4];
        gamma_mu(mu, g);
        const double gs = dagger ? -1.0 : 1.0;
        // forward: (1 - g_mu) s U_mu(x) psi(x+mu)
        {
            int cf[4] = {c[0], c[1], c[2], c[3]};
            cf[mu] = (c[mu] + 1) % G.len(mu);
            const long j = G.idx(cf[0], cf[1], cf[2], cf[3]);
            const double s = (mu == 3 && G.ap && c[3] == G.T - 1) ? -1.0 : 1.0;
            const cd* u = U + (i * 4 + mu) * 9;
            cd w[12]; // U psi
            for (int sp = 0; sp < 4; ++sp) for (int a = 0; a < 3; ++a) {
                cd acc = 0.0;
                for (int b = 0; b < 3; ++b) acc += u[a * 3 + b] * in[j * 12 + sp * 3 + b];
                w[sp * 3 + a] = acc;
            }
            for (int sp = 0; sp < 4; ++sp) for (int a = 0; a < 3; ++a) {
                cd acc = 0.0;
                for (int sq = 0; sq < 4; ++sq) acc += ((sp == sq ? 1.0 : 0.0) - gs * g[sp][sq]) * w[sq * 3 + a];
                out[sp * 3 + a] += s * acc;
            }
        }
        // backward: (1 + g_mu) s U_mu(x-mu)^dag psi(x-mu)
        {
            int cb[4] = {c[0], c[1], c[2], c[3]};
            cb[mu] = (c[mu] + G.len(mu) - 1) % G.len(mu);
            const long j = G.idx(cb[0], cb[1], cb[2], cb[3]);
            const double s = (mu == 3 && G.ap && cb[3] == G.T - 1) ? -1.0 : 1.0;
            const cd* u = U + (j * 4 + mu) * 9;
            cd w[12]; // U^dag psi
            for (int sp = 0; sp < 4; ++sp) for (int a = 0; a < 3; ++a) {
                cd acc = 0.0;
                for (int b = 0; b < 3; ++b) acc += std::conj(u[b * 3 + a]) * in[j * 12 + sp * 3 + b];
                w[sp * 3 + a] = acc;
            }
            for (int sp = 0; sp < 4; ++sp) for (int a = 0; a < 3; ++a) {
                cd acc = 0.0;
                for (int sq = 0; sq < 4; ++sq) acc += ((sp == sq ? 1.0 : 0.0) + gs * g[sp][sq]) * w[sq * 3 + a];
                out[sp * 3 + a] += s * acc;
            }
        }
    }
}

static void hop(const Geom& G, const cd* U, const cd* in, cd* out, int dagger)
{
#pragma omp parallel for schedule(static)
    for (long i = 0; i < G.V; ++i) hop_site(G, U, in, i, dagger, out + i * 12);
}

extern "C" void orc_hop(const int* dims, int ap, const double* U, const double* in, double* out, int dagger)
{
    Geom G(dims, ap);
    hop(G, (const cd*)U, (const cd*)in, (cd*)out, dagger);
}

// single-site evaluation of the same definition from gathered data (for sampled parity at sizes
// where full canonical fields are not held): fwd/bwd links and neighbour spinors are passed in.
//   Ufwd[mu] = U_mu(x), Ubwd[mu] = U_mu(x-mu), nf[mu] = psi(x+mu), nb[mu] = psi(x-mu),
//   sf[mu], sb[mu] = boundary signs of the forward / backward hop.
extern "C" void orc_hop_gathered(const double* Ufwd_, const double* Ubwd_, const double* nf_, const double* nb_,
                                 const double* sf, const double* sb, int dagger, double* out_)
{
    const cd* Ufwd = (const cd*)Ufwd_; const cd* Ubwd = (const cd*)Ubwd_;
    const cd* nf = (const cd*)nf_; const cd* nb = (const cd*)nb_;
    cd* out = (cd*)out_;
    for (int k = 0; k < 12; ++k) out[k] = 0.0;
    const double gs = dagger ? -1.0 : 1.0;
    for (int mu = 0; mu < 4; ++mu) {
        cd g[4][4];
        gamma_mu(mu, g);
        cd w[12], v[12];
        for (int sp = 0; sp < 4; ++sp) for (int a = 0; a < 3; ++a) {
            cd acc = 0.0, acc2 = 0.0;
            for (int b = 0; b < 3; ++b) {
                acc += Ufwd[mu * 9 + a * 3 + b] * nf[mu * 12 + sp * 3 + b];
                acc2 += std::conj(Ubwd[mu * 9 + b * 3 + a]) * nb[mu * 12 + sp * 3 + b];
            }
            w[sp * 3 + a] = acc; v[sp * 3 + a] = acc2;
        }
        for (int sp = 0; sp < 4; ++sp) for (int a = 0; a < 3; ++a) {
            cd acc = 0.0, acc2 = 0.0;
            for (int sq = 0; sq < 4; ++sq) {
                const double d = (sp == sq) ? 1.0 : 0.0;
                acc += (d - gs * g[sp][sq]) * w[sq * 3 + a];
                acc2 += (d + gs * g[sp][sq]) * v[sq * 3 + a];
            }
            out[sp * 3 + a] += sf[mu] * acc + sb[mu] * acc2;
        }
    }
}

// ---------------------------------------------------------------------------------------
// local twist R(a) = 1 + i a g5, a = 2 kappa mu; R^-1 = (1 - i a g5)/(1 + a^2)
// (PAPER.md:162 B = (1 + i 2 kappa mu a g5)^-1; :371-381 "R represents a local twisting operator")
// ---------------------------------------------------------------------------------------
static void twist(const Geom& G, double a, int inverse, const cd* in, cd* out)
{
    cd g5[4][4];
    gamma_mu(4, g5);
    const double nrm = inverse ? 1.0 / (1.0 + a * a) : 1.0;
    const double sa = inverse ? -a : a;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < G.V; ++i)
        for (int sp = 0; sp < 4; ++sp) for (int c = 0; c < 3; ++c) {
            cd acc = in[i * 12 + sp * 3 + c];
            for (int sq = 0; sq < 4; ++sq) acc += I_ * sa * g5[sp][sq] * in[i * 12 + sq * 3 + c];
            out[i * 12 + sp * 3 + c] = nrm * acc;
        }
}

extern "C" void orc_twist(const int* dims, double a, int inverse, const double* in, double* out)
{
    Geom G(dims, 0);
    twist(G, a, inverse, (const cd*)in, (cd*)out);
}

// keep parity p, zero the rest
static void project(const Geom& G, int p, cd* f)
{
#pragma omp parallel for schedule(static)
    for (long i = 0; i < G.V; ++i)
        if (G.parity(i) != p) for (int k = 0; k < 12; ++k) f[i * 12 + k] = 0.0;
}

// full operator M(kappa, mu) psi = psi + i 2 kappa mu g5 psi - kappa Dslash psi; dagger -> M^dag = g5 M(-mu) g5
static void apply_M(const Geom& G, const cd* U, double kappa, double mu, int dagger, const cd* in, cd* out)
{
    std::vector<cd> h(G.V * 12);
    hop(G, U, in, h.data(), dagger);
    const double a = 2.0 * kappa * (dagger ? -mu : mu);
    twist(G, a, 0, in, out);
    for (long k = 0; k < G.V * 12; ++k) out[k] -= kappa * h[k];
}

extern "C" void orc_M(const int* dims, int ap, const double* U, double kappa, double mu, int dagger,
                      const double* in, double* out)
{
    Geom G(dims, ap);
    apply_M(G, (const cd*)U, kappa, mu, dagger, (const cd*)in, (cd*)out);
}

// even-odd preconditioned operator on parity p (asymmetric, PAPER.md:373 Eq. A2 lhs):
//   M_pc = R_pp - kappa^2 Dslash_{p pbar} R_{pbar pbar}^-1 Dslash_{pbar p};  dagger: g_mu -> -g_mu, a -> -a
// `in` is a full-lattice field; only its parity-p part is used; out is zero on parity pbar.
static void apply_Mpc(const Geom& G, const cd* U, double kappa, double mu, int p, int dagger, const cd* in, cd* out)
{
    const double a = 2.0 * kappa * (dagger ? -mu : mu);
    std::vector<cd> v(in, in + G.V * 12), t1(G.V * 12), t2(G.V * 12);
    project(G, p, v.data());
    hop(G, U, v.data(), t1.data(), dagger);    // Dslash_{pbar p} psi_p (lives on pbar)
    project(G, 1 - p, t1.data());
    twist(G, a, 1, t1.data(), t2.data());      // R^-1
    hop(G, U, t2.data(), t1.data(), dagger);   // Dslash_{p pbar}
    project(G, p, t1.data());
    twist(G, a, 0, v.data(), out);             // R psi_p
    for (long k = 0; k < G.V * 12; ++k) out[k] -= kappa * kappa * t1[k];
}

extern "C" void orc_Mpc(const int* dims, int ap, const double* U, double kappa, double mu, int parity, int dagger,
                        const double* in, double* out)
{
    Geom G(dims, ap);
    apply_Mpc(G, (const cd*)U, kappa, mu, parity, dagger, (const cd*)in, (cd*)out);
}

static void apply_MdagM(const Geom& G, const cd* U, double kappa, double mu, int p, const cd* in, cd* out)
{
    std::vector<cd> t(G.V * 12);
    apply_Mpc(G, U, kappa, mu, p, 0, in, t.data());
    apply_Mpc(G, U, kappa, mu, p, 1, t.data(), out);
}

extern "C" void orc_MdagM(const int* dims, int ap, const double* U, double kappa, double mu, int parity,
                          const double* in, double* out)
{
    Geom G(dims, ap);
    apply_MdagM(G, (const cd*)U, kappa, mu, parity, (const cd*)in, (cd*)out);
}

// ---------------------------------------------------------------------------------------
// CG ("the inverter, which is a Conjugate Gradient (CG) solver in this work, is truncated";
// SURVEY.md 8(c-1) items 4-5): solve M s = eta through the even-even Schur system.
//   b'  = eta_e + kappa Dslash_eo R_oo^-1 eta_o
//   b'' = M_pc^dag b'
//   CG on A = M_pc^dag M_pc, x0 = 0, r0 = p0 = b''; stop at the first k with |r_k| <= tol |b''| or k = max_iter
//   s_e = x;  s_o = R_oo^-1 (eta_o + kappa Dslash_oe s_e)
// info[0] = iterations, info[1] = |r_k|/|b''| (iterated), info[2] = |b'' - A x|/|b''| (recomputed),
// info[3] = |eta - M s|/|eta| with the full unpreconditioned operator.
// resid_hist (may be null, length max_iter+1): |r_k|/|b''| per iteration.
// ---------------------------------------------------------------------------------------
static double norm2(const cd* v, long n) { double s = 0; for (long k = 0; k < n; ++k) s += std::norm(v[k]); return s; }
static cd dotc(const cd* a, const cd* b, long n) { cd s = 0; for (long k = 0; k < n; ++k) s += std::conj(a[k]) * b[k]; return s; }

extern "C" void orc_cg_solve(const int* dims, int ap, const double* U_, double kappa, double mu, const double* eta_,
                             double tol, int max_iter, double* s_, double* info, double* resid_hist)
{
    Geom G(dims, ap);
    const cd* U = (const cd*)U_;
    const cd* eta = (const cd*)eta_;
    cd* s = (cd*)s_;
    const long n = G.V * 12;
    const double a = 2.0 * kappa * mu;
    std::vector<cd> eo(eta, eta + n), ee(eta, eta + n), t1(n), t2(n), bp(n), b(n);
    project(G, 1, eo.data());
    project(G, 0, ee.data());
    // b' = eta_e + kappa Dslash_eo R^-1 eta_o
    twist(G, a, 1, eo.data(), t1.data());
    hop(G, U, t1.data(), t2.data(), 0);
    project(G, 0, t2.data());
    for (long k = 0; k < n; ++k) bp[k] = ee[k] + kappa * t2[k];
    // b'' = M_pc^dag b'
    apply_Mpc(G, U, kappa, mu, 0, 1, bp.data(), b.data());
    std::vector<cd> x(n, 0.0), r(b), p(b), Ap(n);
    const double bnorm2 = norm2(b.data(), n);
    double rr = bnorm2;
    int k = 0;
    if (resid_hist) resid_hist[0] = 1.0;
    while (k < max_iter && !(std::sqrt(rr) <= tol * std::sqrt(bnorm2))) {
        apply_MdagM(G, U, kappa, mu, 0, p.data(), Ap.data());
        const double pAp = dotc(p.data(), Ap.data(), n).real();
        const double alpha = rr / pAp;
        for (long q = 0; q < n; ++q) { x[q] += alpha * p[q]; r[q] -= alpha * Ap[q]; }
        const double rr_new = norm2(r.data(), n);
        const double beta = rr_new / rr;
        for (long q = 0; q < n; ++q) p[q] = r[q] + beta * p[q];
        rr = rr_new;
        ++k;
        if (resid_hist) resid_hist[k] = std::sqrt(rr / bnorm2);
    }
    // reconstruct odd sites
    hop(G, U, x.data(), t1.data(), 0);
    project(G, 1, t1.data());
    for (long q = 0; q < n; ++q) t1[q] = eo[q] + kappa * t1[q];
    twist(G, a, 1, t1.data(), t2.data());
    for (long q = 0; q < n; ++q) s[q] = x[q] + t2[q];
    if (info) {
        info[0] = k;
        info[1] = std::sqrt(rr / bnorm2);
        apply_MdagM(G, U, kappa, mu, 0, x.data(), Ap.data());
        for (long q = 0; q < n; ++q) Ap[q] = b[q] - Ap[q];
        info[2] = std::sqrt(norm2(Ap.data(), n) / bnorm2);
        apply_M(G, U, kappa, mu, 0, s, t1.data());
        for (long q = 0; q < n; ++q) t1[q] = eta[q] - t1[q];
        info[3] = std::sqrt(norm2(t1.data(), n) / norm2(eta, n));
    }
}

// ---------------------------------------------------------------------------------------
// loop contraction (PAPER.md:116 Eq. 10; :411 "Traces were taken in color space, leaving the Dirac and
// volume indices open"):  L[n][t] = sum_{x: x4 = t} a(x)^dag (Gamma_n (x) 1_colour) b(x),  n = 0..15
// out[16][T] complex.
// ---------------------------------------------------------------------------------------
extern "C" void orc_loop(const int* dims, const double* a_, const double* b_, double* out_)
{
    Geom G(dims, 0);
    const cd* a = (const cd*)a_;
    const cd* b = (const cd*)b_;
    cd* out = (cd*)out_;
    const long V3 = (long)G.X * G.Y * G.Z;
    for (int n = 0; n < 16; ++n) {
        cd Gm[4][4];
        Gamma_n(n, Gm);
        for (int t = 0; t < G.T; ++t) {
            cd acc = 0.0;
            for (long i = t * V3; i < (t + 1) * V3; ++i)
                for (int al = 0; al < 4; ++al) for (int be = 0; be < 4; ++be) for (int c = 0; c < 3; ++c)
                    acc += std::conj(a[i * 12 + al * 3 + c]) * Gm[al][be] * b[i * 12 + be * 3 + c];
            out[n * G.T + t] = acc;
        }
    }
}
