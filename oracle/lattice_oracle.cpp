// ============================================================================================
// ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// Plain, slow, obviously-correct CPU implementation of the site-parallel lattice-field
// expressions that the CUDA library (include/lqx.h) evaluates.  Only tests/, the smoke check
// in __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may call it.
// It shares NO code with paper_1105_2279_b200/csrc (no headers, helpers, tables, constants).
//
// What it follows.  The paper's method evaluates a QDP++ expression by looping over all lattice
// sites and evaluating the whole expression per site (PAPER.md:61-63 sec.3, :115 sec.5.4); it
// "leaves the data layout, the order of access, the precision of the primitives unchanged"
// (PAPER.md:41).  The method therefore reaches exactly the plain site-by-site definition of
// each expression, and this file IS that definition written out: for every site, fetch the
// operands at the site or at its periodic neighbour, and evaluate with triple loops.
// There is no blocking, fusion, factorisation or reordering.
//
// Layout: external "QDP++ order" (reading A7): site-major array-of-structs, sites
// lexicographic with x0 fastest; inside a site [row][col][re,im] for a colour matrix,
// [spin][colour][re,im] for a fermion, [colour][re,im] for a colour vector, [re,im] complex.
//
// Four instantiations <S storage-in, A arithmetic, O storage-out>:
//   n32 <float , float      , float >  native fp32   (the one that is timed)
//   t32 <float , double     , double>  truth for fp32 configs (inputs fp32, arithmetic fp64)
//   n64 <double, double     , double>  native fp64   (timed)
//   t64 <double, long double, double>  truth for fp64 configs (x87 80-bit arithmetic)
// Reductions accumulate in a type wider than A where one exists (double for float, long double
// otherwise), sequentially in site order, and return double (readings A13).
//
// Compile: g++ -O2 -std=c++17 -ffp-contract=off -fopenmp -shared -fPIC  (see oracle/build.py).
// -ffp-contract=off so results do not depend on the host compiler's FMA choices.
//
// Pins (tests/test_oracle_pins.py, none of them re-types these formulas): unit-gauge staple = 6*1;
// shift round trip; permutation / brute-force neighbour checks; SU(3) products stay unitary;
// gauge invariance of the plaquette and covariance of hop and smear step (the transformation
// is applied with numpy, not with this file); U(1) plane-wave eigenvalue of the hop; point
// source; sum_{x,mu} Re tr[U S^dag] = 4 * plaquette sum; numpy einsum cross-checks on 2^4.
// Jacobi routine (tests/test_jacobi_pins.py): truncated power series of Eq. 2 built with numpy rolls,
// geometric series on unit links, U(1) plane-wave eigenvalue, gauge covariance, iter = 0 / kappa = 0.
// Parity unpinned: nothing -- every exported function has at least one such pin; absolute
// values on the random configs have no printed reference in the paper (there is none).
// ============================================================================================
#include <cstddef>
#include <cstdint>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ------------------------------------------------------------------ O0 geometry (sec. 8a row a1)
// site(x) = x0 + L0*(x1 + L1*(x2 + L2*x3));  nbr(s,sign,mu): x_mu -> (x_mu + sign + L_mu) % L_mu.
// shift(f,FORWARD,mu)(x) = f(x+mu^): fixed by Listing 1 line 25 vs Eq. 2.
struct Geom {
    int L[4];
    long V;
};

Geom make_geom(const int* dims) {
    Geom g;
    g.V = 1;
    for (int d = 0; d < 4; ++d) {
        g.L[d] = dims[d];
        g.V *= dims[d];
    }
    return g;
}

long site_index(const Geom& g, const int x[4]) {
    return x[0] + (long)g.L[0] * (x[1] + (long)g.L[1] * (x[2] + (long)g.L[2] * x[3]));
}

void site_coords(const Geom& g, long s, int x[4]) {
    for (int d = 0; d < 4; ++d) {
        x[d] = (int)(s % g.L[d]);
        s /= g.L[d];
    }
}

long nbr(const Geom& g, long s, int sign, int mu) {
    int x[4];
    site_coords(g, s, x);
    x[mu] = (x[mu] + sign + g.L[mu]) % g.L[mu];
    return site_index(g, x);
}

// ------------------------------------------------------------------ O1 site algebra
template <typename A>
struct Cx {
    A re, im;
};
template <typename A>
Cx<A> operator+(Cx<A> a, Cx<A> b) { return {a.re + b.re, a.im + b.im}; }
template <typename A>
Cx<A> operator-(Cx<A> a, Cx<A> b) { return {a.re - b.re, a.im - b.im}; }
template <typename A>
Cx<A> operator*(Cx<A> a, Cx<A> b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
template <typename A>
Cx<A> conj(Cx<A> a) { return {a.re, -a.im}; }
template <typename A>
Cx<A> scale(A r, Cx<A> a) { return {r * a.re, r * a.im}; }

template <typename A>
struct Mat {
    Cx<A> e[3][3];
};
template <typename A>
struct Vec {
    Cx<A> e[3];
};

// (AB)_ij = sum_k A_ik B_kj, k ascending
template <typename A>
Mat<A> mul(const Mat<A>& a, const Mat<A>& b) {
    Mat<A> c;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            Cx<A> acc = a.e[i][0] * b.e[0][j];
            for (int k = 1; k < 3; ++k) acc = acc + a.e[i][k] * b.e[k][j];
            c.e[i][j] = acc;
        }
    return c;
}
// adj(A)_ij = conj(A_ji)
template <typename A>
Mat<A> adj(const Mat<A>& a) {
    Mat<A> c;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c.e[i][j] = conj(a.e[j][i]);
    return c;
}
template <typename A>
Mat<A> add(const Mat<A>& a, const Mat<A>& b) {
    Mat<A> c;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c.e[i][j] = a.e[i][j] + b.e[i][j];
    return c;
}
template <typename A>
Mat<A> sub(const Mat<A>& a, const Mat<A>& b) {
    Mat<A> c;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c.e[i][j] = a.e[i][j] - b.e[i][j];
    return c;
}
template <typename A>
Mat<A> rscale(A r, const Mat<A>& a) {
    Mat<A> c;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c.e[i][j] = scale(r, a.e[i][j]);
    return c;
}
template <typename A>
Cx<A> trace(const Mat<A>& a) {
    return a.e[0][0] + a.e[1][1] + a.e[2][2];
}
// (Mv)_i = sum_j M_ij v_j, j ascending
template <typename A>
Vec<A> mul(const Mat<A>& m, const Vec<A>& v) {
    Vec<A> w;
    for (int i = 0; i < 3; ++i) {
        Cx<A> acc = m.e[i][0] * v.e[0];
        for (int j = 1; j < 3; ++j) acc = acc + m.e[i][j] * v.e[j];
        w.e[i] = acc;
    }
    return w;
}
template <typename A>
Vec<A> add(const Vec<A>& a, const Vec<A>& b) {
    Vec<A> c;
    for (int i = 0; i < 3; ++i) c.e[i] = a.e[i] + b.e[i];
    return c;
}

// QDP-order loads / stores.  CM real index ((s*3+i)*3+j)*2+c; vectors ((s*nspin+a)*3+i)*2+c.
template <typename A, typename S>
Mat<A> load_mat(const S* f, long s) {
    Mat<A> m;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            m.e[i][j].re = (A)f[((s * 3 + i) * 3 + j) * 2 + 0];
            m.e[i][j].im = (A)f[((s * 3 + i) * 3 + j) * 2 + 1];
        }
    return m;
}
template <typename A, typename O>
void store_mat(O* f, long s, const Mat<A>& m) {
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            f[((s * 3 + i) * 3 + j) * 2 + 0] = (O)m.e[i][j].re;
            f[((s * 3 + i) * 3 + j) * 2 + 1] = (O)m.e[i][j].im;
        }
}
template <typename A, typename S>
Vec<A> load_vec(const S* f, long s, int nspin, int a) {
    Vec<A> v;
    for (int i = 0; i < 3; ++i) {
        v.e[i].re = (A)f[((s * nspin + a) * 3 + i) * 2 + 0];
        v.e[i].im = (A)f[((s * nspin + a) * 3 + i) * 2 + 1];
    }
    return v;
}
template <typename A, typename O>
void store_vec(O* f, long s, int nspin, int a, const Vec<A>& v) {
    for (int i = 0; i < 3; ++i) {
        f[((s * nspin + a) * 3 + i) * 2 + 0] = (O)v.e[i].re;
        f[((s * nspin + a) * 3 + i) * 2 + 1] = (O)v.e[i].im;
    }
}

// Accumulator wider than the arithmetic type where one exists (A13).
template <typename A>
struct Wide {
    typedef long double type;
};
template <>
struct Wide<float> {
    typedef double type;
};

// ------------------------------------------------------------------ O2 shift (row a3)
// out(x) = in(x + sign*mu^); nreal = reals per site.  Pure copy: bit-exact.
template <typename S>
void shift_field(const Geom& g, int nreal, const S* in, S* out, int sign, int mu) {
#pragma omp parallel for schedule(static)
    for (long s = 0; s < g.V; ++s) {
        long n = nbr(g, s, sign, mu);
        for (int r = 0; r < nreal; ++r) out[s * nreal + r] = in[n * nreal + r];
    }
}

// ------------------------------------------------------------------ O3 catalogue (rows a4, a5)
// form (i)  R = A*B + C*adj(D)           (BASELINE.json configs[4])
template <typename S, typename A, typename O>
void mm_plus_madj(const Geom& g, const S* a, const S* b, const S* c, const S* d, O* r) {
#pragma omp parallel for schedule(static)
    for (long s = 0; s < g.V; ++s) {
        Mat<A> ab = mul(load_mat<A>(a, s), load_mat<A>(b, s));
        Mat<A> cd = mul(load_mat<A>(c, s), adj(load_mat<A>(d, s)));
        store_mat(r, s, add(ab, cd));
    }
}
// form (ii) c = trace(A*B) -> LatticeComplex
template <typename S, typename A, typename O>
void trace_mm(const Geom& g, const S* a, const S* b, O* c) {
#pragma omp parallel for schedule(static)
    for (long s = 0; s < g.V; ++s) {
        Cx<A> t = trace(mul(load_mat<A>(a, s), load_mat<A>(b, s)));
        c[s * 2 + 0] = (O)t.re;
        c[s * 2 + 1] = (O)t.im;
    }
}
// form (iii) R = alpha*A - shift(B, sign, mu); alpha rounded once to the storage precision (A10)
template <typename S, typename A, typename O>
void ax_minus_shift(const Geom& g, double alpha, const S* a, const S* b, int sign, int mu, O* r) {
    const A al = (A)(S)alpha;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < g.V; ++s) {
        Mat<A> t = sub(rscale(al, load_mat<A>(a, s)), load_mat<A>(b, nbr(g, s, sign, mu)));
        store_mat(r, s, t);
    }
}
// form (iv) w = M*v, per spin component (nspin = 1 colour vector, 4 fermion)
template <typename S, typename A, typename O>
void mat_vec(const Geom& g, int nspin, const S* m, const S* v, O* w) {
#pragma omp parallel for schedule(static)
    for (long s = 0; s < g.V; ++s) {
        Mat<A> mm = load_mat<A>(m, s);
        for (int a = 0; a < nspin; ++a) store_vec(w, s, nspin, a, mul(mm, load_vec<A>(v, s, nspin, a)));
    }
}
// E3 of Listing 1 (reading A3): r = s0 + kappa*h ; any field kind, ncx complex/site
template <typename S, typename A, typename O>
void axpy(const Geom& g, int ncx, const S* s0, double kappa, const S* h, O* r) {
    const A k = (A)(S)kappa;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < g.V * ncx * 2; ++i) r[i] = (O)((A)s0[i] + k * (A)h[i]);
}
// r = sc * a   (catalogue real-scalar scaling)
template <typename S, typename A, typename O>
void scale_field(const Geom& g, int ncx, double sc, const S* a, O* r) {
    const A k = (A)(S)sc;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < g.V * ncx * 2; ++i) r[i] = (O)(k * (A)a[i]);
}
// E4 of Listing 1: chi /= norm -- a true division (reading A22)
template <typename S, typename A, typename O>
void divide_field(const Geom& g, int ncx, double nrm, const S* a, O* r) {
    const A k = (A)(S)nrm;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < g.V * ncx * 2; ++i) r[i] = (O)((A)a[i] / k);
}

// ------------------------------------------------------------------ hop (row a6)
// chi(x) = sum_{mu=0..3} U_mu(x) psi(x+mu^) + adj(U_mu(x-mu^)) psi(x-mu^)
// (BASELINE.json configs[1]; = Listing 1 line 25/27 summed over mu; Eq. 2 :215)
template <typename S, typename A, typename O>
void hop(const Geom& g, int nspin, const S* const u[4], const S* psi, O* chi) {
#pragma omp parallel for schedule(static)
    for (long s = 0; s < g.V; ++s) {
        for (int a = 0; a < nspin; ++a) {
            Vec<A> acc;
            for (int mu = 0; mu < 4; ++mu) {
                long f = nbr(g, s, +1, mu), b = nbr(g, s, -1, mu);
                Vec<A> fw = mul(load_mat<A>(u[mu], s), load_vec<A>(psi, f, nspin, a));
                Vec<A> bw = mul(adj(load_mat<A>(u[mu], b)), load_vec<A>(psi, b, nspin, a));
                Vec<A> t = add(fw, bw);
                acc = (mu == 0) ? t : add(acc, t);
            }
            store_vec(chi, s, nspin, a, acc);
        }
    }
}
// The same expression evaluated literally as Listing 1 writes it, with the temporary it implies:
// tmp = adj(u[mu])*psi (site-local) then shift(tmp,BACKWARD,mu).  Used only as a pin (bit-for-bit
// equal to hop()).
template <typename S, typename A, typename O>
void hop_listing(const Geom& g, int nspin, const S* const u[4], const S* psi, O* chi) {
    std::vector<Vec<A>> tmp((size_t)g.V * nspin), acc((size_t)g.V * nspin);
    for (int mu = 0; mu < 4; ++mu) {
        for (long s = 0; s < g.V; ++s)
            for (int a = 0; a < nspin; ++a)
                tmp[s * nspin + a] = mul(adj(load_mat<A>(u[mu], s)), load_vec<A>(psi, s, nspin, a));
        for (long s = 0; s < g.V; ++s)
            for (int a = 0; a < nspin; ++a) {
                Vec<A> fw = mul(load_mat<A>(u[mu], s), load_vec<A>(psi, nbr(g, s, +1, mu), nspin, a));
                Vec<A> t = add(fw, tmp[nbr(g, s, -1, mu) * nspin + a]);
                acc[s * nspin + a] = (mu == 0) ? t : add(acc[s * nspin + a], t);
            }
    }
    for (long s = 0; s < g.V; ++s)
        for (int a = 0; a < nspin; ++a) store_vec(chi, s, nspin, a, acc[s * nspin + a]);
}

// ------------------------------------------------------------------ Jacobi smearing
// Listing 1 of the paper, step by step in its order (readings A2, A3):
//   s_0 = chi                                                        (line 16, E0)
//   for n = 0 .. iter-1:
//       psi = chi                                                    (line 20, E0)
//       for mu = 0 .. Nd-1, mu != no_smear_dir:
//           first mu :  h_smear  = u[mu]*shift(psi,FORWARD,mu) + shift(adj(u[mu])*psi,BACKWARD,mu)   (line 25, E1)
//           later mu :  h_smear += (the same expression)                                             (line 27, E2)
//       chi = s_0 + kappa * h_smear                                  (line 30, E3)
//   chi /= norm                                                      (line 33, E4)
// which is the power series sum_{n<=iter} kappa^n H^n s_0 / norm of the inverse of K, Eq. 2.
// Intermediate fields are kept in the arithmetic type A (for the native instantiations A is the storage
// type, as in a QDP++ build of that precision; for the truth instantiations nothing is rounded on the way).
template <typename S, typename A, typename O>
void jacobi_smear(const Geom& g, int nspin, const S* const u[4], const S* chi_in, double kappa, int iter, int no_smear_dir,
                  double norm, O* chi_out) {
    const size_t n = (size_t)g.V * nspin;
    std::vector<Vec<A>> s0(n), chi(n), psi(n), h(n);
    for (long s = 0; s < g.V; ++s)
        for (int a = 0; a < nspin; ++a) s0[s * nspin + a] = chi[s * nspin + a] = load_vec<A>(chi_in, s, nspin, a);
    const A k = (A)(S)kappa, nrm = (A)(S)norm;
    for (int it = 0; it < iter; ++it) {
        psi = chi;
        bool first = true;
        for (int mu = 0; mu < 4; ++mu) {
            if (mu == no_smear_dir) continue;
#pragma omp parallel for schedule(static)
            for (long s = 0; s < g.V; ++s) {
                const long f = nbr(g, s, +1, mu), b = nbr(g, s, -1, mu);
                const Mat<A> uf = load_mat<A>(u[mu], s), ub = adj(load_mat<A>(u[mu], b));
                for (int a = 0; a < nspin; ++a) {
                    const Vec<A> t = add(mul(uf, psi[f * nspin + a]), mul(ub, psi[b * nspin + a]));
                    h[s * nspin + a] = first ? t : add(h[s * nspin + a], t);
                }
            }
            first = false;
        }
#pragma omp parallel for schedule(static)
        for (long i = 0; i < (long)n; ++i)
            for (int c = 0; c < 3; ++c) {
                const Cx<A> hh = first ? Cx<A>{(A)0, (A)0} : h[i].e[c];  // every direction excluded: h_smear = 0
                chi[i].e[c].re = s0[i].e[c].re + k * hh.re;
                chi[i].e[c].im = s0[i].e[c].im + k * hh.im;
            }
    }
    for (long s = 0; s < g.V; ++s)
        for (int a = 0; a < nspin; ++a) {
            Vec<A> v = chi[s * nspin + a];
            for (int c = 0; c < 3; ++c) {
                v.e[c].re = v.e[c].re / nrm;
                v.e[c].im = v.e[c].im / nrm;
            }
            store_vec(chi_out, s, nspin, a, v);
        }
}

// ------------------------------------------------------------------ O4 reductions (row a9)
// sum(f): one site object; out[2*ncx] doubles in QDP order.
template <typename S, typename A>
void sum_field(const Geom& g, int ncx, const S* f, double* out) {
    typedef typename Wide<A>::type W;
    std::vector<W> acc(2 * ncx, (W)0);
    for (long s = 0; s < g.V; ++s)
        for (int r = 0; r < 2 * ncx; ++r) acc[r] += (W)f[s * 2 * ncx + r];
    for (int r = 0; r < 2 * ncx; ++r) out[r] = (double)acc[r];
}
// norm2(f) = sum_x sum_components |c|^2
template <typename S, typename A>
double norm2_field(const Geom& g, int ncx, const S* f) {
    typedef typename Wide<A>::type W;
    W acc = 0;
    for (long i = 0; i < g.V * 2 * ncx; ++i) acc += (W)f[i] * (W)f[i];
    return (double)acc;
}
// trace as a global reduction: sum_x tr M(x) (reading A12)
template <typename S, typename A>
void trace_field(const Geom& g, const S* m, double out[2]) {
    typedef typename Wide<A>::type W;
    W re = 0, im = 0;
    for (long s = 0; s < g.V; ++s)
        for (int i = 0; i < 3; ++i) {
            re += (W)m[((s * 3 + i) * 3 + i) * 2 + 0];
            im += (W)m[((s * 3 + i) * 3 + i) * 2 + 1];
        }
    out[0] = (double)re;
    out[1] = (double)im;
}

// ------------------------------------------------------------------ O6 plaquette (row a8)
// P = sum_x sum_{mu<nu} Re tr[ U_mu(x) U_nu(x+mu^) adj(U_mu(x+nu^)) adj(U_nu(x)) ]
template <typename S, typename A>
A plaquette_site(const Geom& g, const S* const u[4], long s) {
    A p = 0;
    for (int mu = 0; mu < 4; ++mu)
        for (int nu = mu + 1; nu < 4; ++nu) {
            Mat<A> m = mul(load_mat<A>(u[mu], s), load_mat<A>(u[nu], nbr(g, s, +1, mu)));
            m = mul(m, adj(load_mat<A>(u[mu], nbr(g, s, +1, nu))));
            m = mul(m, adj(load_mat<A>(u[nu], s)));
            p += trace(m).re;
        }
    return p;
}
template <typename S, typename A>
double plaquette_sum(const Geom& g, const S* const u[4]) {
    typedef typename Wide<A>::type W;
    std::vector<A> per_site((size_t)g.V);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < g.V; ++s) per_site[s] = plaquette_site<S, A>(g, u, s);
    W acc = 0;
    for (long s = 0; s < g.V; ++s) acc += (W)per_site[s];
    return (double)acc;
}

// ------------------------------------------------------------------ O5 staple sum + smear (row a7)
// S_mu(x) = sum_{nu != mu} [ U_nu(x) U_mu(x+nu^) adj(U_nu(x+mu^))
//                          + adj(U_nu(x-nu^)) U_mu(x-nu^) U_nu(x-nu^+mu^) ]      (configs[0])
// nu ascending, upper then lower, products left to right.
template <typename S, typename A>
Mat<A> staple_sum_site(const Geom& g, const S* const u[4], long s, int mu) {
    Mat<A> acc;
    bool first = true;
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        long xpnu = nbr(g, s, +1, nu), xpmu = nbr(g, s, +1, mu), xmnu = nbr(g, s, -1, nu);
        long xmnupmu = nbr(g, xmnu, +1, mu);
        Mat<A> up = mul(mul(load_mat<A>(u[nu], s), load_mat<A>(u[mu], xpnu)), adj(load_mat<A>(u[nu], xpmu)));
        Mat<A> lo = mul(mul(adj(load_mat<A>(u[nu], xmnu)), load_mat<A>(u[mu], xmnu)), load_mat<A>(u[nu], xmnupmu));
        acc = first ? up : add(acc, up);
        acc = add(acc, lo);
        first = false;
    }
    return acc;
}
// U'_mu(x) = (1-a) U_mu(x) + (a/6) S_mu(x); both coefficients computed in double and rounded once
// to the storage precision (reading A10).  No projection back to SU(3) (reading A9).
template <typename S, typename A>
Mat<A> smear_link(const Geom& g, const S* const u[4], double alpha, long s, int mu) {
    const A c0 = (A)(S)(1.0 - alpha), c1 = (A)(S)(alpha / 6.0);
    return add(rscale(c0, load_mat<A>(u[mu], s)), rscale(c1, staple_sum_site<S, A>(g, u, s, mu)));
}
template <typename S, typename A, typename O>
void staple_sum(const Geom& g, const S* const u[4], int mu, O* out) {
#pragma omp parallel for schedule(static)
    for (long s = 0; s < g.V; ++s) store_mat(out, s, staple_sum_site<S, A>(g, u, s, mu));
}
template <typename S, typename A, typename O>
void smear_step(const Geom& g, const S* const uin[4], double alpha, O* const uout[4]) {
    for (int mu = 0; mu < 4; ++mu) {
#pragma omp parallel for schedule(static)
        for (long s = 0; s < g.V; ++s) store_mat(uout[mu], s, smear_link<S, A>(g, uin, alpha, s, mu));
    }
}
// the same, for a list of (site, mu) samples: out[n][18] -- for full-size parity on sampled links
template <typename S, typename A, typename O>
void smear_links(const Geom& g, const S* const uin[4], double alpha, long n, const long* sites,
                 const int* mus, O* out) {
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; ++k) store_mat(out, k, smear_link<S, A>(g, uin, alpha, sites[k], mus[k]));
}
// per-site plaquette values for a list of sites (sampled check of the plaquette integrand)
template <typename S, typename A>
void plaquette_sites(const Geom& g, const S* const u[4], long n, const long* sites, double* out) {
#pragma omp parallel for schedule(static)
    for (long k = 0; k < n; ++k) out[k] = (double)plaquette_site<S, A>(g, u, sites[k]);
}

}  // namespace

// ============================================================================================
// C entry points (ctypes).  Suffix = instantiation.
// ============================================================================================
extern "C" {

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
long orc_site_index(const int* dims, const int* x) { return site_index(make_geom(dims), x); }
void orc_site_coords(const int* dims, long s, int* x) { site_coords(make_geom(dims), s, x); }
void orc_neighbor_table(const int* dims, int sign, int mu, int32_t* out) {
    Geom g = make_geom(dims);
    for (long s = 0; s < g.V; ++s) out[s] = (int32_t)nbr(g, s, sign, mu);
}
void orc_shift_f32(const int* dims, int nreal, const float* in, float* out, int sign, int mu) {
    shift_field(make_geom(dims), nreal, in, out, sign, mu);
}
void orc_shift_f64(const int* dims, int nreal, const double* in, double* out, int sign, int mu) {
    shift_field(make_geom(dims), nreal, in, out, sign, mu);
}

#define ORC_INSTANTIATE(SUF, S, A, O)                                                                      \
    void orc_mm_plus_madj_##SUF(const int* dims, const S* a, const S* b, const S* c, const S* d, O* r) {   \
        mm_plus_madj<S, A, O>(make_geom(dims), a, b, c, d, r);                                             \
    }                                                                                                      \
    void orc_trace_mm_##SUF(const int* dims, const S* a, const S* b, O* c) {                               \
        trace_mm<S, A, O>(make_geom(dims), a, b, c);                                                       \
    }                                                                                                      \
    void orc_ax_minus_shift_##SUF(const int* dims, double alpha, const S* a, const S* b, int sign, int mu, \
                                  O* r) {                                                                  \
        ax_minus_shift<S, A, O>(make_geom(dims), alpha, a, b, sign, mu, r);                                \
    }                                                                                                      \
    void orc_mat_vec_##SUF(const int* dims, int nspin, const S* m, const S* v, O* w) {                     \
        mat_vec<S, A, O>(make_geom(dims), nspin, m, v, w);                                                 \
    }                                                                                                      \
    void orc_axpy_##SUF(const int* dims, int ncx, const S* s0, double kappa, const S* h, O* r) {           \
        axpy<S, A, O>(make_geom(dims), ncx, s0, kappa, h, r);                                              \
    }                                                                                                      \
    void orc_scale_##SUF(const int* dims, int ncx, double sc, const S* a, O* r) {                          \
        scale_field<S, A, O>(make_geom(dims), ncx, sc, a, r);                                              \
    }                                                                                                      \
    void orc_divide_##SUF(const int* dims, int ncx, double nrm, const S* a, O* r) {                        \
        divide_field<S, A, O>(make_geom(dims), ncx, nrm, a, r);                                            \
    }                                                                                                      \
    void orc_hop_##SUF(const int* dims, int nspin, const S* u0, const S* u1, const S* u2, const S* u3,     \
                       const S* psi, O* chi) {                                                             \
        const S* u[4] = {u0, u1, u2, u3};                                                                  \
        hop<S, A, O>(make_geom(dims), nspin, u, psi, chi);                                                 \
    }                                                                                                      \
    void orc_hop_listing_##SUF(const int* dims, int nspin, const S* u0, const S* u1, const S* u2,          \
                               const S* u3, const S* psi, O* chi) {                                        \
        const S* u[4] = {u0, u1, u2, u3};                                                                  \
        hop_listing<S, A, O>(make_geom(dims), nspin, u, psi, chi);                                         \
    }                                                                                                      \
    void orc_jacobi_smear_##SUF(const int* dims, int nspin, const S* u0, const S* u1, const S* u2,         \
                                const S* u3, const S* chi, double kappa, int iter, int no_smear_dir,       \
                                double norm, O* out) {                                                     \
        const S* u[4] = {u0, u1, u2, u3};                                                                  \
        jacobi_smear<S, A, O>(make_geom(dims), nspin, u, chi, kappa, iter, no_smear_dir, norm, out);       \
    }                                                                                                      \
    void orc_sum_##SUF(const int* dims, int ncx, const S* f, double* out) {                                \
        sum_field<S, A>(make_geom(dims), ncx, f, out);                                                     \
    }                                                                                                      \
    double orc_norm2_##SUF(const int* dims, int ncx, const S* f) {                                         \
        return norm2_field<S, A>(make_geom(dims), ncx, f);                                                 \
    }                                                                                                      \
    void orc_trace_##SUF(const int* dims, const S* m, double* out) {                                       \
        trace_field<S, A>(make_geom(dims), m, out);                                                        \
    }                                                                                                      \
    double orc_plaquette_sum_##SUF(const int* dims, const S* u0, const S* u1, const S* u2, const S* u3) {  \
        const S* u[4] = {u0, u1, u2, u3};                                                                  \
        return plaquette_sum<S, A>(make_geom(dims), u);                                                    \
    }                                                                                                      \
    void orc_plaquette_sites_##SUF(const int* dims, const S* u0, const S* u1, const S* u2, const S* u3,    \
                                   long n, const long* sites, double* out) {                               \
        const S* u[4] = {u0, u1, u2, u3};                                                                  \
        plaquette_sites<S, A>(make_geom(dims), u, n, sites, out);                                          \
    }                                                                                                      \
    void orc_staple_sum_##SUF(const int* dims, const S* u0, const S* u1, const S* u2, const S* u3, int mu, \
                              O* out) {                                                                    \
        const S* u[4] = {u0, u1, u2, u3};                                                                  \
        staple_sum<S, A, O>(make_geom(dims), u, mu, out);                                                  \
    }                                                                                                      \
    void orc_smear_step_##SUF(const int* dims, const S* u0, const S* u1, const S* u2, const S* u3,         \
                              double alpha, O* r0, O* r1, O* r2, O* r3) {                                  \
        const S* u[4] = {u0, u1, u2, u3};                                                                  \
        O* r[4] = {r0, r1, r2, r3};                                                                        \
        smear_step<S, A, O>(make_geom(dims), u, alpha, r);                                                 \
    }                                                                                                      \
    void orc_smear_links_##SUF(const int* dims, const S* u0, const S* u1, const S* u2, const S* u3,        \
                               double alpha, long n, const long* sites, const int* mus, O* out) {          \
        const S* u[4] = {u0, u1, u2, u3};                                                                  \
        smear_links<S, A, O>(make_geom(dims), u, alpha, n, sites, mus, out);                               \
    }

ORC_INSTANTIATE(n32, float, float, float)
ORC_INSTANTIATE(t32, float, double, double)
ORC_INSTANTIATE(n64, double, double, double)
ORC_INSTANTIATE(t64, double, long double, double)

}  // extern "C"
