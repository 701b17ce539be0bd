// ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// Plain, slow, FP64 CPU implementation of what the hot path of arxiv 2407.09700 computes:
// contracted four-centre ERIs (Eq. 1-5) digested with a density matrix into J and K
// (Alg. 2 lines 8-13 read as full sums) and the J/K nuclear gradient
// (Eq. 12-15, prefactors per SURVEY.md 8(c) R10).
//
// The paper's method (Rys quadrature) reaches these textbook quantities exactly, so the oracle is the
// plain definition evaluated by a DIFFERENT algorithm: McMurchie-Davidson (paper ref. 10) with a
// directly evaluated Boys function.  No Rys roots, no tables, no permutational symmetry, no screening
// unless explicitly asked for.  It shares no code, header, table or constant with the CUDA path.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
//
// Conventions: primitives are the raw Cartesian Gaussians of Eq. 2; coefficients
// multiply the raw primitive; spherical functions are obtained from the contracted Cartesian block with
// the matrices handed in through oracle_set_c2s (built in oracle/sph.py by a route independent of the
// library).  Cartesian component order inside a shell: lx descending, then ly descending.
//
// Pins (tests/test_oracle_*.py): closed-form (ss|ss) with erf, F_m against the incomplete gamma function
// and mpmath quadrature, Gauss-Hermite x Gauss-Legendre brute-force quadrature of primitive ERIs up to
// g functions, centre-derivative ladder, 8-fold symmetry, translational invariance, J/K symmetry and
// linearity, R9 symmetry-list digestion == plain quadruple loop, gradient per-axis sums = 0 and central
// finite differences of E_J, E_K; the contraction loop and the four-index Cartesian -> spherical transform for l >= 1
// against contracted blocks assembled from brute-force quadrature components (test_contracted_spherical_block_vs_quadrature);
// orthonormality of contracted spherical shells through the E_0 overlap (test_contracted_spherical_shells_are_orthonormal).  Absolute J/K/gradient values on the synthetic clusters have no
// external reference ("parity unpinned" beyond this chain).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int LMAX = 6;          // i (capacity only: array bounds, no arithmetic depends on it)
constexpr int LTOT_MAX = 4 * LMAX + 1;  // 25 with one raised index (gradient)

struct Shell { int32_t atom, l, nprim, prim_off, ao_off; };
struct Prim { double e, c; };

struct BasisView {
  const Shell* sh; int nsh; const Prim* pr; int npr; const double* xyz; int natm; int nao;
};

inline int ncart(int l) { return (l + 1) * (l + 2) / 2; }
inline int nsph(int l) { return 2 * l + 1; }

// c2s[l] : ns(l) x nc(l), row-major, spherical index m=-l..l.  Set from Python (oracle/sph.py).
std::vector<double> g_c2s[LMAX + 1];

// ------------------------------------------------------------------------------------------------
// Boys function F_m(x) = int_0^1 t^(2m) exp(-x t^2) dt, evaluated directly.
// x < 35: ascending series for the highest m (all terms positive), then downward recursion
//         F_{m-1} = (2x F_m + e^-x) / (2m-1).
// x >= 35: F_0 = sqrt(pi/x)/2 * erf(sqrt x), upward recursion F_{m+1} = ((2m+1) F_m - e^-x) / (2x).
void boys(int mmax, double x, double* F) {
  if (x < 35.0) {
    const double ex = std::exp(-x);
    double term = 1.0 / (2 * mmax + 1);
    double sum = term;
    for (int i = 1; i < 400; ++i) {
      term *= 2.0 * x / (2 * mmax + 2 * i + 1);
      sum += term;
      if (term < 1e-18 * sum) break;
    }
    F[mmax] = ex * sum;
    for (int m = mmax; m > 0; --m) F[m - 1] = (2.0 * x * F[m] + ex) / (2 * m - 1);
  } else {
    const double ex = std::exp(-x);
    F[0] = 0.5 * std::sqrt(M_PI / x) * std::erf(std::sqrt(x));
    for (int m = 0; m < mmax; ++m) F[m + 1] = ((2 * m + 1) * F[m] - ex) / (2.0 * x);
  }
}

// ------------------------------------------------------------------------------------------------
// Hermite expansion coefficients for one axis:
//   E_0^{00} = exp(-mu X_AB^2)
//   E_t^{i+1,j} = E_{t-1}^{ij}/(2p) + (P-A) E_t^{ij} + (t+1) E_{t+1}^{ij}
//   E_t^{i,j+1} = E_{t-1}^{ij}/(2p) + (P-B) E_t^{ij} + (t+1) E_{t+1}^{ij}
// stored as E[(i*(lb+1)+j)*(la+lb+1)+t].
void hermite_E(int la, int lb, double a, double b, double A, double B, std::vector<double>& E) {
  const double p = a + b, mu = a * b / p, P = (a * A + b * B) / p;
  const int nt = la + lb + 1;
  E.assign((size_t)(la + 1) * (lb + 1) * nt, 0.0);
  auto at = [&](int i, int j, int t) -> double& { return E[((size_t)i * (lb + 1) + j) * nt + t]; };
  auto get = [&](int i, int j, int t) -> double { return (t < 0 || t > i + j) ? 0.0 : at(i, j, t); };
  at(0, 0, 0) = std::exp(-mu * (A - B) * (A - B));
  for (int i = 0; i <= la; ++i) {
    if (i > 0)
      for (int t = 0; t <= i; ++t)
        at(i, 0, t) = get(i - 1, 0, t - 1) / (2 * p) + (P - A) * get(i - 1, 0, t) + (t + 1) * get(i - 1, 0, t + 1);
    for (int j = 1; j <= lb; ++j)
      for (int t = 0; t <= i + j; ++t)
        at(i, j, t) = get(i, j - 1, t - 1) / (2 * p) + (P - B) * get(i, j - 1, t) + (t + 1) * get(i, j - 1, t + 1);
  }
}

// One "function" of a primitive pair: three 1-D Hermite coefficient strings (x,y,z).
struct Fun { const double* e[3]; int n[3]; };

struct PrimPair {
  double p, P[3], cc, ea;           // p = a+b, centre, c_a*c_b, exponent of the first function
  std::vector<double> E[3];         // per axis, for angular momenta (la_eff, lb)
};

struct PairData {
  int la, lb, la_eff;               // la_eff = la+1 when the first index is to be differentiated
  std::vector<PrimPair> pp;
};

void make_pair(const BasisView& bv, int i, int j, int raise, PairData& out) {
  const Shell& si = bv.sh[i]; const Shell& sj = bv.sh[j];
  out.la = si.l; out.lb = sj.l; out.la_eff = si.l + raise;
  out.pp.clear();
  const double* A = bv.xyz + 3 * si.atom; const double* B = bv.xyz + 3 * sj.atom;
  for (int ka = 0; ka < si.nprim; ++ka)
    for (int kb = 0; kb < sj.nprim; ++kb) {
      const Prim& pa = bv.pr[si.prim_off + ka]; const Prim& pb = bv.pr[sj.prim_off + kb];
      PrimPair q; q.p = pa.e + pb.e; q.cc = pa.c * pb.c; q.ea = pa.e;
      for (int x = 0; x < 3; ++x) {
        q.P[x] = (pa.e * A[x] + pb.e * B[x]) / q.p;
        hermite_E(out.la_eff, out.lb, pa.e, pb.e, A[x], B[x], q.E[x]);
      }
      out.pp.push_back(std::move(q));
    }
}

inline void cart_powers(int l, int idx, int* pw) {  // lx descending, then ly descending
  int c = 0;
  for (int lx = l; lx >= 0; --lx)
    for (int ly = l - lx; ly >= 0; --ly) { if (c == idx) { pw[0] = lx; pw[1] = ly; pw[2] = l - lx - ly; return; } ++c; }
}

struct Scratch {
  std::vector<double> R;   // R[n][t][u][v]
  std::vector<double> W;   // W[t][u][v]
  std::vector<double> dE;  // derivative Hermite strings
  std::vector<double> cart, tmp1, tmp2;
};

// Hermite Coulomb integrals: R^(n)_000 = (-2a)^n F_n(a |PQ|^2),
// R^(n)_{t+1,u,v} = t R^(n+1)_{t-1,u,v} + X_PQ R^(n+1)_{tuv} (same in u, v).  On return R0 = R^(0) in a cube of side L+1.
void hermite_R(int L, double alpha, const double* PQ, std::vector<double>& R) {
  const int S = L + 1;
  R.assign((size_t)S * S * S * S, 0.0);
  auto at = [&](int n, int t, int u, int v) -> double& { return R[(((size_t)n * S + t) * S + u) * S + v]; };
  double F[LTOT_MAX + 2];
  const double r2 = PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2];
  boys(L, alpha * r2, F);
  double f = 1.0;
  for (int n = 0; n <= L; ++n) { at(n, 0, 0, 0) = f * F[n]; f *= -2.0 * alpha; }
  for (int k = 1; k <= L; ++k)             // total order t+u+v
    for (int n = 0; n <= L - k; ++n)
      for (int t = 0; t <= k; ++t)
        for (int u = 0; u <= k - t; ++u) {
          const int v = k - t - u;
          double val;
          if (t > 0)      val = (t > 1 ? (t - 1) * at(n + 1, t - 2, u, v) : 0.0) + PQ[0] * at(n + 1, t - 1, u, v);
          else if (u > 0) val = (u > 1 ? (u - 1) * at(n + 1, t, u - 2, v) : 0.0) + PQ[1] * at(n + 1, t, u - 1, v);
          else            val = (v > 1 ? (v - 1) * at(n + 1, t, u, v - 2) : 0.0) + PQ[2] * at(n + 1, t, u, v - 1);
          at(n, t, u, v) = val;
        }
}

// Primitive quartet:
// [f|g] = 2 pi^{5/2}/(p q sqrt(p+q)) sum_{tuv} E^f_t E^f_u E^f_v sum_{tau nu phi} (-1)^{tau+nu+phi} E^g_tau E^g_nu E^g_phi R_{t+tau,u+nu,v+phi}
// out[f*nket+g] += scale * [f|g]
void prim_quartet(const Fun* bra, int nbra, int Lbra, const Fun* ket, int nket, int Lket,
                  double p, const double* P, double q, const double* Q, double scale, double* out, Scratch& s) {
  const int L = Lbra + Lket, S = L + 1, SB = Lbra + 1;
  const double alpha = p * q / (p + q);
  const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
  hermite_R(L, alpha, PQ, s.R);
  const double* R0 = s.R.data();  // n = 0 slab
  const double pref = scale * 2.0 * std::pow(M_PI, 2.5) / (p * q * std::sqrt(p + q));
  s.W.resize((size_t)SB * SB * SB);
  for (int g = 0; g < nket; ++g) {
    const Fun& kf = ket[g];
    for (int t = 0; t <= Lbra; ++t)
      for (int u = 0; u <= Lbra - t; ++u)
        for (int v = 0; v <= Lbra - t - u; ++v) {
          double w = 0.0;
          for (int a = 0; a < kf.n[0]; ++a)
            for (int b = 0; b < kf.n[1]; ++b)
              for (int c = 0; c < kf.n[2]; ++c) {
                const double sgn = ((a + b + c) & 1) ? -1.0 : 1.0;
                w += sgn * kf.e[0][a] * kf.e[1][b] * kf.e[2][c] * R0[((size_t)(t + a) * S + (u + b)) * S + (v + c)];
              }
          s.W[((size_t)t * SB + u) * SB + v] = w;
        }
    for (int f = 0; f < nbra; ++f) {
      const Fun& bf = bra[f];
      double acc = 0.0;
      for (int t = 0; t < bf.n[0]; ++t)
        for (int u = 0; u < bf.n[1]; ++u)
          for (int v = 0; v < bf.n[2]; ++v)
            acc += bf.e[0][t] * bf.e[1][u] * bf.e[2][v] * s.W[((size_t)t * SB + u) * SB + v];
      out[(size_t)f * nket + g] += pref * acc;
    }
  }
}

// Build the function list of a primitive pair for plain (deriv<0) or differentiated (first index, all 3 axes) shells.
// Derivative of a raw primitive on its own centre (Eq. 2): d/dA_x [a] = 2 alpha [a+1_x] - a_x [a-1_x].
void build_funs(const PairData& pd, const PrimPair& pp, bool deriv, std::vector<Fun>& funs, std::vector<double>& dE) {
  const int la = pd.la, lb = pd.lb, le = pd.la_eff, nt = le + lb + 1;
  const int na = ncart(la), nb = ncart(lb);
  auto str = [&](int x, int i, int j) { return pp.E[x].data() + ((size_t)i * (lb + 1) + j) * nt; };
  funs.clear();
  if (!deriv) {
    for (int ia = 0; ia < na; ++ia)
      for (int ib = 0; ib < nb; ++ib) {
        int pa[3], pb[3]; cart_powers(la, ia, pa); cart_powers(lb, ib, pb);
        Fun f;
        for (int x = 0; x < 3; ++x) { f.e[x] = str(x, pa[x], pb[x]); f.n[x] = pa[x] + pb[x] + 1; }
        funs.push_back(f);
      }
    return;
  }
  // derivative strings: dE[x][ia][ib][t]
  dE.assign((size_t)3 * na * nb * nt, 0.0);
  for (int x = 0; x < 3; ++x)
    for (int ia = 0; ia < na; ++ia)
      for (int ib = 0; ib < nb; ++ib) {
        int pa[3], pb[3]; cart_powers(la, ia, pa); cart_powers(lb, ib, pb);
        double* d = dE.data() + (((size_t)x * na + ia) * nb + ib) * nt;
        const double* up = str(x, pa[x] + 1, pb[x]);
        for (int t = 0; t <= pa[x] + 1 + pb[x]; ++t) d[t] = 2.0 * pp.ea * up[t];
        if (pa[x] > 0) {
          const double* dn = str(x, pa[x] - 1, pb[x]);
          for (int t = 0; t <= pa[x] - 1 + pb[x]; ++t) d[t] -= pa[x] * dn[t];
        }
      }
  for (int x = 0; x < 3; ++x)       // f = x*(na*nb) + ia*nb + ib
    for (int ia = 0; ia < na; ++ia)
      for (int ib = 0; ib < nb; ++ib) {
        int pa[3], pb[3]; cart_powers(la, ia, pa); cart_powers(lb, ib, pb);
        Fun f;
        for (int y = 0; y < 3; ++y) {
          if (y == x) { f.e[y] = dE.data() + (((size_t)x * na + ia) * nb + ib) * nt; f.n[y] = pa[y] + pb[y] + 2; }
          else        { f.e[y] = str(y, pa[y], pb[y]); f.n[y] = pa[y] + pb[y] + 1; }
        }
        funs.push_back(f);
      }
}

// transform index `which` (0..3 of a [d0][d1][d2][d3] row-major block, with nlead leading copies) by T (ns x nc)
void transform_index(const double* in, double* out, int nlead, const int* dims, int which, const double* T, int ns) {
  int pre = nlead, post = 1;
  for (int i = 0; i < which; ++i) pre *= dims[i];
  for (int i = which + 1; i < 4; ++i) post *= dims[i];
  const int nc = dims[which];
  for (int a = 0; a < pre; ++a)
    for (int s = 0; s < ns; ++s)
      for (int b = 0; b < post; ++b) {
        double acc = 0.0;
        for (int c = 0; c < nc; ++c) acc += T[(size_t)s * nc + c] * in[((size_t)a * nc + c) * post + b];
        out[((size_t)a * ns + s) * post + b] = acc;
      }
}

// Contracted spherical block (ij|kl) (Eq. 5 then c2s), or the three first-index derivative blocks if deriv.
// out: [nlead][ns_i][ns_j][ns_k][ns_l], nlead = deriv ? 3 : 1.
void shell_quartet(const PairData& bra, const PairData& ket, bool deriv, double* out, Scratch& s) {
  const int la = bra.la, lb = bra.lb, lc = ket.la, ld = ket.lb;
  const int nbra = (deriv ? 3 : 1) * ncart(la) * ncart(lb), nket = ncart(lc) * ncart(ld);
  s.cart.assign((size_t)nbra * nket, 0.0);
  std::vector<Fun> bf, kf; std::vector<double> dEk;
  const int Lbra = la + lb + (deriv ? 1 : 0), Lket = lc + ld;
  for (const PrimPair& pb : bra.pp) {
    build_funs(bra, pb, deriv, bf, s.dE);
    for (const PrimPair& pk : ket.pp) {
      build_funs(ket, pk, false, kf, dEk);
      prim_quartet(bf.data(), nbra, Lbra, kf.data(), nket, Lket, pb.p, pb.P, pk.p, pk.P, pb.cc * pk.cc, s.cart.data(), s);
    }
  }
  // Cartesian -> spherical on all four indices
  const int nlead = deriv ? 3 : 1;
  int dims[4] = {ncart(la), ncart(lb), ncart(lc), ncart(ld)};
  const int ls[4] = {la, lb, lc, ld};
  std::vector<double>* cur = &s.cart; std::vector<double>* nxt = &s.tmp1;
  for (int w = 0; w < 4; ++w) {
    size_t sz = nlead; for (int i = 0; i < 4; ++i) sz *= (i == w ? nsph(ls[i]) : dims[i]);
    nxt->resize(sz);
    transform_index(cur->data(), nxt->data(), nlead, dims, w, g_c2s[ls[w]].data(), nsph(ls[w]));
    dims[w] = nsph(ls[w]);
    cur = nxt; nxt = (cur == &s.tmp1) ? &s.tmp2 : &s.tmp1;
  }
  std::memcpy(out, cur->data(), sizeof(double) * (size_t)nlead * dims[0] * dims[1] * dims[2] * dims[3]);
}

BasisView view(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm) {
  BasisView bv; bv.sh = reinterpret_cast<const Shell*>(shells); bv.nsh = nsh;
  bv.pr = reinterpret_cast<const Prim*>(prims); bv.npr = npr; bv.xyz = xyz; bv.natm = natm;
  bv.nao = 0; for (int i = 0; i < nsh; ++i) bv.nao = std::max(bv.nao, bv.sh[i].ao_off + nsph(bv.sh[i].l));
  return bv;
}

struct PairTable {   // all ordered pairs (k,l), plain (not raised)
  int nsh; std::vector<PairData> t;
  void build(const BasisView& bv) {
    nsh = bv.nsh; t.resize((size_t)nsh * nsh);
#pragma omp parallel for schedule(dynamic, 16)
    for (long kl = 0; kl < (long)nsh * nsh; ++kl) make_pair(bv, (int)(kl / nsh), (int)(kl % nsh), 0, t[kl]);
  }
  const PairData& operator()(int k, int l) const { return t[(size_t)k * nsh + l]; }
};

void schwarz_matrix(const BasisView& bv, const PairTable& pt, std::vector<double>& Q) {
  const int n = bv.nsh; Q.assign((size_t)n * n, 0.0);
#pragma omp parallel
  {
    Scratch s; std::vector<double> blk;
#pragma omp for schedule(dynamic, 8)
    for (long ij = 0; ij < (long)n * n; ++ij) {
      const int i = (int)(ij / n), j = (int)(ij % n);
      if (j > i) continue;
      const int ni = nsph(bv.sh[i].l), nj = nsph(bv.sh[j].l);
      blk.resize((size_t)ni * nj * ni * nj);
      shell_quartet(pt(i, j), pt(i, j), false, blk.data(), s);
      double m = 0.0;
      for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
        m = std::max(m, std::fabs(blk[(((size_t)a * nj + b) * ni + a) * nj + b]));
      Q[(size_t)i * n + j] = Q[(size_t)j * n + i] = std::sqrt(m);
    }
  }
}

}  // namespace

extern "C" {

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}

// c2s matrix for angular momentum l: ns(l) x nc(l), row-major.
int oracle_set_c2s(int l, const double* T) {
  if (l < 0 || l > LMAX) return -1;
  g_c2s[l].assign(T, T + (size_t)nsph(l) * ncart(l));
  return 0;
}

void oracle_boys(int mmax, double x, double* F) { boys(mmax, x, F); }

// Single primitive Cartesian ERI [ab|cd] over raw Gaussians (Eq. 2), powers pw[4][3], exponents ex[4], centres ctr[4][3].
double oracle_prim_eri(const int* pw, const double* ex, const double* ctr) {
  std::vector<double> E[2][3];
  Fun f[2]; double p[2], P[2][3];
  for (int s = 0; s < 2; ++s) {
    const int* pa = pw + 6 * s; const int* pb = pa + 3;
    const double a = ex[2 * s], b = ex[2 * s + 1];
    const double* A = ctr + 6 * s; const double* B = A + 3;
    p[s] = a + b;
    for (int x = 0; x < 3; ++x) {
      P[s][x] = (a * A[x] + b * B[x]) / p[s];
      hermite_E(pa[x], pb[x], a, b, A[x], B[x], E[s][x]);
      f[s].e[x] = E[s][x].data() + ((size_t)pa[x] * (pb[x] + 1) + pb[x]) * (pa[x] + pb[x] + 1);
      f[s].n[x] = pa[x] + pb[x] + 1;
    }
  }
  int Lb = 0, Lk = 0;
  for (int x = 0; x < 3; ++x) { Lb += pw[x] + pw[3 + x]; Lk += pw[6 + x] + pw[9 + x]; }
  Scratch s; double out = 0.0;
  prim_quartet(&f[0], 1, Lb, &f[1], 1, Lk, p[0], P[0], p[1], P[1], 1.0, &out, s);
  return out;
}

// Spherical block (ij|kl): out[ns_i][ns_j][ns_k][ns_l]; deriv!=0: out[3][...] = d/dR_{atom(i)} acting on function i only.
void oracle_eri_block(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm,
                      int i, int j, int k, int l, int deriv, double* out) {
  BasisView bv = view(shells, nsh, prims, npr, xyz, natm);
  PairData bra, ket; make_pair(bv, i, j, deriv ? 1 : 0, bra); make_pair(bv, k, l, 0, ket);
  Scratch s; shell_quartet(bra, ket, deriv != 0, out, s);
}

// Overlap block <i|j> of two contracted spherical shells from the E_0 Hermite coefficients (SURVEY 8(c) table "c2s matrices"):
// S = sum_prims c_a c_b E_0^x E_0^y E_0^z (pi/p)^{3/2}, then the same index transform as shell_quartet on indices 0 and 1.
// A pin helper: shells normalised by reading R2 must give the unit matrix for i == j.  out: [ns_i][ns_j].
void oracle_overlap_block(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm,
                          int i, int j, double* out) {
  BasisView bv = view(shells, nsh, prims, npr, xyz, natm);
  PairData pd; make_pair(bv, i, j, 0, pd);
  const int la = pd.la, lb = pd.lb, na = ncart(la), nb = ncart(lb), nt = la + lb + 1;
  std::vector<double> cart((size_t)na * nb, 0.0), half((size_t)nsph(la) * nb), full((size_t)nsph(la) * nsph(lb));
  for (const PrimPair& pp : pd.pp)
    for (int ia = 0; ia < na; ++ia)
      for (int ib = 0; ib < nb; ++ib) {
        int pa[3], pb[3]; cart_powers(la, ia, pa); cart_powers(lb, ib, pb);
        double e0 = 1.0;
        for (int x = 0; x < 3; ++x) e0 *= pp.E[x][((size_t)pa[x] * (lb + 1) + pb[x]) * nt];
        cart[(size_t)ia * nb + ib] += pp.cc * e0 * std::pow(M_PI / pp.p, 1.5);
      }
  int dims[4] = {na, nb, 1, 1};
  transform_index(cart.data(), half.data(), 1, dims, 0, g_c2s[la].data(), nsph(la));
  dims[0] = nsph(la);
  transform_index(half.data(), full.data(), 1, dims, 1, g_c2s[lb].data(), nsph(lb));
  std::memcpy(out, full.data(), sizeof(double) * full.size());
}

// Schwarz factors Q_ij = max over spherical components |(ab|ab)|^(1/2) (Eq. 7).  Q: [nsh][nsh].
void oracle_schwarz(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm, double* Q) {
  BasisView bv = view(shells, nsh, prims, npr, xyz, natm);
  PairTable pt; pt.build(bv);
  std::vector<double> q; schwarz_matrix(bv, pt, q);
  std::memcpy(Q, q.data(), sizeof(double) * q.size());
}

// J_ij = sum_kl (ij|kl) D_kl,  K_ik = sum_jl (ij|kl) D_jl : plain loop over ALL ordered shell quartets.
// thr > 0: "same screening" mode, skips exactly the quartets with Q_ij Q_kl < thr (reading R7), Q from this oracle.
// Returns the number of shell quartets evaluated.
// group_of != nullptr: density-weighted screening of the paper (Eq. 8-9) at the level of shell groups:
// a quartet is skipped iff Q_ij Q_kl min(1, P) < thr with P = max |D| over the six sub-blocks of D between the shell groups
// of i, j, k, l (the groups are the caller's: shells of equal angular momentum and contraction degree).
// The cap at 1 makes the density factor only ever remove quartets from the Schwarz-only list.
static long long jk_loop(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm,
                         const double* D, double thr, const int32_t* group_of, int ng, double* J, double* K) {
  BasisView bv = view(shells, nsh, prims, npr, xyz, natm);
  const int nao = bv.nao;
  PairTable pt; pt.build(bv);
  std::vector<double> Q; if (thr > 0) schwarz_matrix(bv, pt, Q);
  std::vector<double> Pg;   // Pg[ga][gb] = max |D_mu,nu|, mu in a shell of group ga, nu in a shell of group gb
  if (group_of) {
    Pg.assign((size_t)ng * ng, 0.0);
    for (int a = 0; a < nsh; ++a)
      for (int b = 0; b < nsh; ++b)
        for (int m = 0; m < nsph(bv.sh[a].l); ++m)
          for (int n = 0; n < nsph(bv.sh[b].l); ++n) {
            double& p = Pg[(size_t)group_of[a] * ng + group_of[b]];
            p = std::max(p, std::fabs(D[(size_t)(bv.sh[a].ao_off + m) * nao + bv.sh[b].ao_off + n]));
          }
  }
  auto dens_factor = [&](int i, int j, int k, int l) {
    if (!group_of) return 1.0;
    const int g[4] = {group_of[i], group_of[j], group_of[k], group_of[l]};
    double P = 0.0;
    for (int x = 0; x < 4; ++x) for (int y = 0; y < 4; ++y) if (x != y) P = std::max(P, Pg[(size_t)g[x] * ng + g[y]]);
    return std::min(1.0, P);
  };
  std::fill(J, J + (size_t)nao * nao, 0.0); std::fill(K, K + (size_t)nao * nao, 0.0);
  long long count = 0;
#pragma omp parallel reduction(+ : count)
  {
    Scratch s; std::vector<double> blk; std::vector<double> Kp((size_t)nao * nao, 0.0);
#pragma omp for schedule(dynamic, 1)
    for (long ij = 0; ij < (long)nsh * nsh; ++ij) {
      const int i = (int)(ij / nsh), j = (int)(ij % nsh);
      const Shell& si = bv.sh[i]; const Shell& sj = bv.sh[j];
      const int ni = nsph(si.l), nj = nsph(sj.l);
      for (int k = 0; k < nsh; ++k)
        for (int l = 0; l < nsh; ++l) {
          if (thr > 0 && Q[(size_t)i * nsh + j] * Q[(size_t)k * nsh + l] * dens_factor(i, j, k, l) < thr) continue;
          const Shell& sk = bv.sh[k]; const Shell& sl = bv.sh[l];
          const int nk = nsph(sk.l), nl = nsph(sl.l);
          blk.resize((size_t)ni * nj * nk * nl);
          shell_quartet(pt(i, j), pt(k, l), false, blk.data(), s);
          ++count;
          size_t e = 0;
          for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
            for (int c = 0; c < nk; ++c) for (int d = 0; d < nl; ++d, ++e) {
              const double g = blk[e];
              // J_ij row is owned by this (i,j) iteration: no race
              J[(size_t)(si.ao_off + a) * nao + sj.ao_off + b] += g * D[(size_t)(sk.ao_off + c) * nao + sl.ao_off + d];
              Kp[(size_t)(si.ao_off + a) * nao + sk.ao_off + c] += g * D[(size_t)(sj.ao_off + b) * nao + sl.ao_off + d];
            }
        }
    }
#pragma omp critical
    for (size_t x = 0; x < (size_t)nao * nao; ++x) K[x] += Kp[x];
  }
  return count;
}

long long oracle_jk(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm,
                    const double* D, double thr, double* J, double* K) {
  return jk_loop(shells, nsh, prims, npr, xyz, natm, D, thr, nullptr, 0, J, K);
}

long long oracle_jk_dscreen(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm,
                            const double* D, double thr, const int32_t* group_of, int ng, double* J, double* K) {
  return jk_loop(shells, nsh, prims, npr, xyz, natm, D, thr, group_of, ng, J, K);
}

// Block mode for large systems: Jblk for shell pairs (i,j) = sum over all (k,l); Kblk for shell pairs (i,k) = sum over all (j,l).
// pairs: [n][2]; out: concatenated row-major blocks ns_first x ns_second.
void oracle_j_blocks(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm,
                     const double* D, const int32_t* pairs, int npairs, double* out) {
  BasisView bv = view(shells, nsh, prims, npr, xyz, natm);
  const int nao = bv.nao;
  PairTable pt; pt.build(bv);
  size_t off = 0;
  for (int ip = 0; ip < npairs; ++ip) {
    const int i = pairs[2 * ip], j = pairs[2 * ip + 1];
    const Shell& si = bv.sh[i]; const Shell& sj = bv.sh[j];
    const int ni = nsph(si.l), nj = nsph(sj.l);
    std::vector<double> acc((size_t)ni * nj, 0.0);
#pragma omp parallel
    {
      Scratch s; std::vector<double> blk, loc((size_t)ni * nj, 0.0);
#pragma omp for schedule(dynamic, 4)
      for (long kl = 0; kl < (long)nsh * nsh; ++kl) {
        const int k = (int)(kl / nsh), l = (int)(kl % nsh);
        const Shell& sk = bv.sh[k]; const Shell& sl = bv.sh[l];
        const int nk = nsph(sk.l), nl = nsph(sl.l);
        blk.resize((size_t)ni * nj * nk * nl);
        shell_quartet(pt(i, j), pt(k, l), false, blk.data(), s);
        size_t e = 0;
        for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
          for (int c = 0; c < nk; ++c) for (int d = 0; d < nl; ++d, ++e)
            loc[(size_t)a * nj + b] += blk[e] * D[(size_t)(sk.ao_off + c) * nao + sl.ao_off + d];
      }
#pragma omp critical
      for (size_t x = 0; x < loc.size(); ++x) acc[x] += loc[x];
    }
    std::memcpy(out + off, acc.data(), sizeof(double) * acc.size()); off += acc.size();
  }
}

void oracle_k_blocks(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm,
                     const double* D, const int32_t* pairs, int npairs, double* out) {
  BasisView bv = view(shells, nsh, prims, npr, xyz, natm);
  const int nao = bv.nao;
  PairTable pt; pt.build(bv);
  size_t off = 0;
  for (int ip = 0; ip < npairs; ++ip) {
    const int i = pairs[2 * ip], k = pairs[2 * ip + 1];
    const Shell& si = bv.sh[i]; const Shell& sk = bv.sh[k];
    const int ni = nsph(si.l), nk = nsph(sk.l);
    std::vector<double> acc((size_t)ni * nk, 0.0);
#pragma omp parallel
    {
      Scratch s; std::vector<double> blk, loc((size_t)ni * nk, 0.0);
#pragma omp for schedule(dynamic, 4)
      for (long jl = 0; jl < (long)nsh * nsh; ++jl) {
        const int j = (int)(jl / nsh), l = (int)(jl % nsh);
        const Shell& sj = bv.sh[j]; const Shell& sl = bv.sh[l];
        const int nj = nsph(sj.l), nl = nsph(sl.l);
        blk.resize((size_t)ni * nj * nk * nl);
        shell_quartet(pt(i, j), pt(k, l), false, blk.data(), s);
        size_t e = 0;
        for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
          for (int c = 0; c < nk; ++c) for (int d = 0; d < nl; ++d, ++e)
            loc[(size_t)a * nk + c] += blk[e] * D[(size_t)(sj.ao_off + b) * nao + sl.ao_off + d];
      }
#pragma omp critical
      for (size_t x = 0; x < loc.size(); ++x) acc[x] += loc[x];
    }
    std::memcpy(out + off, acc.data(), sizeof(double) * acc.size()); off += acc.size();
  }
}

// Explicit quartet list (cfg1): every listed shell quartet (i,j,k,l) adds its six updates once
// (Alg. 2 lines 8-13), no symmetry factor, no final symmetrisation:
//  Jt_ij += g D_kl, Jt_kl += g D_ij, Kt_ik += g D_jl, Kt_jl += g D_ik, Kt_il += g D_jk, Kt_jk += g D_il.
void oracle_digest_list(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm,
                        const double* D, const int32_t* quartets, int nq, double* Jt, double* Kt) {
  BasisView bv = view(shells, nsh, prims, npr, xyz, natm);
  const int nao = bv.nao;
  std::fill(Jt, Jt + (size_t)nao * nao, 0.0); std::fill(Kt, Kt + (size_t)nao * nao, 0.0);
#pragma omp parallel
  {
    Scratch s; std::vector<double> blk, Jp((size_t)nao * nao, 0.0), Kp((size_t)nao * nao, 0.0);
    PairData bra, ket;
#pragma omp for schedule(dynamic, 8)
    for (int iq = 0; iq < nq; ++iq) {
      const int i = quartets[4 * iq], j = quartets[4 * iq + 1], k = quartets[4 * iq + 2], l = quartets[4 * iq + 3];
      make_pair(bv, i, j, 0, bra); make_pair(bv, k, l, 0, ket);
      const Shell& si = bv.sh[i]; const Shell& sj = bv.sh[j]; const Shell& sk = bv.sh[k]; const Shell& sl = bv.sh[l];
      const int ni = nsph(si.l), nj = nsph(sj.l), nk = nsph(sk.l), nl = nsph(sl.l);
      blk.resize((size_t)ni * nj * nk * nl);
      shell_quartet(bra, ket, false, blk.data(), s);
      size_t e = 0;
      for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
        for (int c = 0; c < nk; ++c) for (int d = 0; d < nl; ++d, ++e) {
          const double g = blk[e];
          const size_t ia = si.ao_off + a, jb = sj.ao_off + b, kc = sk.ao_off + c, ld = sl.ao_off + d;
          Jp[ia * nao + jb] += g * D[kc * nao + ld];
          Jp[kc * nao + ld] += g * D[ia * nao + jb];
          Kp[ia * nao + kc] += g * D[jb * nao + ld];
          Kp[jb * nao + ld] += g * D[ia * nao + kc];
          Kp[ia * nao + ld] += g * D[jb * nao + kc];
          Kp[jb * nao + kc] += g * D[ia * nao + ld];
        }
    }
#pragma omp critical
    for (size_t x = 0; x < (size_t)nao * nao; ++x) { Jt[x] += Jp[x]; Kt[x] += Kp[x]; }
  }
}

// J/K nuclear gradient at fixed D (Eq. 12-15 with the prefactors of reading R10):
//   gradJ[A,x] = 2 sum_{a in A} sum_{bcd} D_ab D_cd (d_x a b|cd),  gradK[A,x] = 2 sum_{a in A} sum_{bcd} D_ac D_bd (d_x a b|cd)
// for E_J = 1/2 sum D_ij D_kl (ij|kl), E_K = 1/2 sum D_ik D_jl (ij|kl); sums over ALL ordered quartets.
// atoms: list of atoms whose rows are wanted (natoms_sel<=0: all).  Rows of other atoms are left zero ("row mode").
// thr > 0 skips quartets with Q_ij Q_kl < thr.
void oracle_jk_grad(const int32_t* shells, int nsh, const double* prims, int npr, const double* xyz, int natm,
                    const double* D, const int32_t* atoms, int natoms_sel, double thr, double* gradJ, double* gradK) {
  BasisView bv = view(shells, nsh, prims, npr, xyz, natm);
  const int nao = bv.nao;
  PairTable pt; pt.build(bv);
  std::vector<double> Q; if (thr > 0) schwarz_matrix(bv, pt, Q);
  std::vector<char> want(natm, natoms_sel <= 0 ? 1 : 0);
  for (int x = 0; x < natoms_sel; ++x) want[atoms[x]] = 1;
  std::fill(gradJ, gradJ + 3 * natm, 0.0); std::fill(gradK, gradK + 3 * natm, 0.0);
#pragma omp parallel
  {
    Scratch s; std::vector<double> blk; PairData bra;
    std::vector<double> gJ(3 * natm, 0.0), gK(3 * natm, 0.0);
#pragma omp for schedule(dynamic, 1)
    for (long ij = 0; ij < (long)nsh * nsh; ++ij) {
      const int i = (int)(ij / nsh), j = (int)(ij % nsh);
      const Shell& si = bv.sh[i]; const Shell& sj = bv.sh[j];
      if (!want[si.atom]) continue;
      make_pair(bv, i, j, 1, bra);
      const int ni = nsph(si.l), nj = nsph(sj.l);
      for (int k = 0; k < nsh; ++k)
        for (int l = 0; l < nsh; ++l) {
          if (thr > 0 && Q[(size_t)i * nsh + j] * Q[(size_t)k * nsh + l] < thr) continue;
          const Shell& sk = bv.sh[k]; const Shell& sl = bv.sh[l];
          const int nk = nsph(sk.l), nl = nsph(sl.l);
          const size_t nb = (size_t)ni * nj * nk * nl;
          blk.resize(3 * nb);
          shell_quartet(bra, pt(k, l), true, blk.data(), s);
          for (int x = 0; x < 3; ++x) {
            size_t e = x * nb; double aj = 0.0, ak = 0.0;
            for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
              for (int c = 0; c < nk; ++c) for (int d = 0; d < nl; ++d, ++e) {
                const size_t ia = si.ao_off + a, jb = sj.ao_off + b, kc = sk.ao_off + c, ld = sl.ao_off + d;
                aj += blk[e] * D[ia * nao + jb] * D[kc * nao + ld];
                ak += blk[e] * D[ia * nao + kc] * D[jb * nao + ld];
              }
            gJ[3 * si.atom + x] += 2.0 * aj; gK[3 * si.atom + x] += 2.0 * ak;
          }
        }
    }
#pragma omp critical
    for (int x = 0; x < 3 * natm; ++x) { gradJ[x] += gJ[x]; gradK[x] += gK[x]; }
  }
}

}  // extern "C"
