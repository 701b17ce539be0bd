// generic.cu -- reference-path kernels of liberi_b200: run-time angular momenta (l <= 4 each, any order), one thread per
// shell quartet, 2-D integrals of one Rys root at a time in per-thread local memory.  Correctness first: this is the
// path every tuned kernel is checked against, the one behind eri_compute_quartets / eri_schwarz, and the fallback for
// classes without a tuned kernel.  Structure follows the paper's Algorithm 3: per primitive
// quartet, roots -> 2-D integrals -> product over the three axes (Eq. 1) -> digestion before contraction
// (PAPER.md:125).  The recurrences are those of DESIGN.md reading R5 (the paper does not print them).
#include "eri_dev.cuh"
#include "launch.h"

namespace eri {
namespace {

// Capacity of the per-thread local arrays: LC = 4 serves every input up to g (625 words per axis and root); LC = 6 is the
// h/i instantiation (2401 words per axis: 58 KB of local memory per thread -- the footprint the paper names as its limit,
// PAPER.md:151; only launched when a unit really contains an h or i shell).
template <int LC> struct Cap {
  static constexpr int G = (LC + 1) * (LC + 1) * (LC + 1) * (LC + 1);        // plain 2-D integrals of one axis
  static constexpr int G1 = (LC + 2) * (LC + 2) * (LC + 2) * (LC + 1);       // raised on a, b, c (gradient)
  static constexpr int NM = 2 * LC + 3;                                      // nmax + 1 with both bra indices raised
  static constexpr int NR = (4 * LC + 1) / 2 + 1;                            // roots, gradient included
};

struct QuartetGeom {
  double A[3], AB[3], C[3], CD[3];
  int la, lb, lc, ld;
};

// 2-D integrals I(i,j,k,l) of one axis for one root (reading R5):
//   I(0,0)=init; I(n+1,m) = C00 I(n,m) + n B10 I(n-1,m) + m B00 I(n,m-1); I(n,m+1) = C00' I(n,m) + m B01 I(n,m-1) + n B00 I(n-1,m)
//   I(i,j+1,k,l) = I(i+1,j,k,l) + (A-B) I(i,j,k,l);  I(i,j,k,l+1) = I(i,j,k+1,l) + (C-D) I(i,j,k,l)
// dims of the result: [na][nb][nc][nd] with na = la+1 (+raise) etc.; nmax = na+nb-2, mmax = nc+nd-2.
// Numerical hygiene: the recurrence is built on the centre of the pair that is NEARER to
// the product centre P (the one with the larger exponent) and transferred to the other one; the opposite order loses
// up to (|AB|/|PB|)^l digits when a tight and a diffuse function sit several Bohr apart.  swap_bra: build on B,
// transfer to A with (B-A); c00 must then be given relative to B.  Same for the ket.
template <int LC>
__device__ void fill_2d(double* __restrict__ G, int na, int nb, int nc, int nd, double init, double c00, double c00p,
                        double b10, double b01, double b00, double ab, double cd, bool swap_bra, bool swap_ket) {
  const int nmax = na + nb - 2, mmax = nc + nd - 2, M1 = mmax + 1;
  double T0[Cap<LC>::NM * Cap<LC>::NM];   // up to (l+1 raised): nmax, mmax <= 2 LC + 2
  double tmp[Cap<LC>::NM * (LC + 2)];
  double Bm[(LC + 2) * (LC + 2) * Cap<LC>::NM];
  T0[0] = init;
  for (int n = 0; n < nmax; ++n) T0[(n + 1) * M1] = c00 * T0[n * M1] + (n > 0 ? n * b10 * T0[(n - 1) * M1] : 0.0);
  for (int m = 0; m < mmax; ++m)
    for (int n = 0; n <= nmax; ++n) {
      double v = c00p * T0[n * M1 + m];
      if (m > 0) v += m * b01 * T0[n * M1 + m - 1];
      if (n > 0) v += n * b00 * T0[(n - 1) * M1 + m];
      T0[n * M1 + m + 1] = v;
    }
  // bra transfer: n1 = dimension of the centre the recurrence was built on, n2 = the other one
  const int n1 = swap_bra ? nb : na, n2 = swap_bra ? na : nb;
  const double x12 = swap_bra ? -ab : ab;
  for (int m = 0; m <= mmax; ++m) {
    for (int i = 0; i <= nmax; ++i) tmp[i * n2] = T0[i * M1 + m];
    for (int j = 1; j < n2; ++j)
      for (int i = 0; i <= nmax - j; ++i) tmp[i * n2 + j] = tmp[(i + 1) * n2 + j - 1] + x12 * tmp[i * n2 + j - 1];
    for (int i = 0; i < n1; ++i)
      for (int j = 0; j < n2; ++j) Bm[(swap_bra ? j * nb + i : i * nb + j) * M1 + m] = tmp[i * n2 + j];
  }
  // ket transfer
  const int m1 = swap_ket ? nd : nc, m2 = swap_ket ? nc : nd;
  const double y12 = swap_ket ? -cd : cd;
  for (int ij = 0; ij < na * nb; ++ij) {
    for (int k = 0; k <= mmax; ++k) tmp[k * m2] = Bm[ij * M1 + k];
    for (int l = 1; l < m2; ++l)
      for (int k = 0; k <= mmax - l; ++k) tmp[k * m2 + l] = tmp[(k + 1) * m2 + l - 1] + y12 * tmp[k * m2 + l - 1];
    for (int k = 0; k < m1; ++k)
      for (int l = 0; l < m2; ++l) G[ij * nc * nd + (swap_ket ? l * nd + k : k * nd + l)] = tmp[k * m2 + l];
  }
}

// true if the second centre of the pair (B = A - AB) is nearer to the product centre P than the first one
__device__ __forceinline__ bool swap_centre(const double* P, const double* A, const double* AB) {
  double da = 0.0, db = 0.0;
  for (int x = 0; x < 3; ++x) { const double pa = P[x] - A[x], pb = pa + AB[x]; da += pa * pa; db += pb * pb; }
  return db < da;
}

// work item -> (bra pair i, ket pair j, weight); false if the thread has nothing to do
__device__ __forceinline__ bool locate(const Work& w, int& i, int& j, double& f) {
  const int blk = blockIdx.x * w.nshard + w.shard;
  if (w.list) {
    const long t = (long)blk * (blockDim.x * blockDim.y) + threadIdx.y * blockDim.x + threadIdx.x;
    if (t >= w.nlist) return false;
    i = w.list[t].x; j = w.list[t].y; f = 1.0;
    return true;
  }
  if (blk >= w.row_off[w.nrows]) return false;
  const int r = find_row(w.row_off, w.nrows, blk);
  const int jb = blk - w.row_off[r];
  i = r * blockDim.y + threadIdx.y;
  j = jb * blockDim.x + threadIdx.x;
  if (i >= w.bra.npair) return false;
  if (j >= w.ket_count[i]) return false;
  f = w.bra.geom[6 * w.bra.stride + i] * w.ket.geom[6 * w.ket.stride + j];
  if (w.same && i == j) f *= 0.5;
  return true;
}

__device__ __forceinline__ void load_geom(const Work& w, int i, int j, QuartetGeom& g) {
  const PairSet& b = w.bra; const PairSet& k = w.ket;
  for (int x = 0; x < 3; ++x) {
    g.A[x] = b.geom[x * b.stride + i]; g.AB[x] = b.geom[(3 + x) * b.stride + i];
    g.C[x] = k.geom[x * k.stride + j]; g.CD[x] = k.geom[(3 + x) * k.stride + j];
  }
  g.la = b.la; g.lb = b.lb; g.lc = k.la; g.ld = k.lb;
}

// Loop over primitive quartets and roots; after the three 2-D integral arrays of a root are ready call
// cons(gx, gy, gz) -- the weight and all prefactors are folded into gz.
template <int LC, typename Consumer>
__device__ void quartet_loop(const Work& w, int i, int j, const QuartetGeom& g, Consumer& cons, int kb_first = 0, int kb_step = 1) {
  const PairSet& b = w.bra; const PairSet& k = w.ket;
  const int N = nroots_of(g.la + g.lb + g.lc + g.ld);
  const int na = g.la + 1, nb = g.lb + 1, nc = g.lc + 1, nd = g.ld + 1;
  double gx[Cap<LC>::G], gy[Cap<LC>::G], gz[Cap<LC>::G];
  double u[Cap<LC>::NR], wt[Cap<LC>::NR];
  for (int kb = kb_first; kb < b.npp; kb += kb_step) {
    const double p = b.prim[(kb * 5 + 0) * b.stride + i];
    const double P[3] = {b.prim[(kb * 5 + 1) * b.stride + i], b.prim[(kb * 5 + 2) * b.stride + i], b.prim[(kb * 5 + 3) * b.stride + i]};
    const double Kab = b.prim[(kb * 5 + 4) * b.stride + i];
    for (int kk = 0; kk < k.npp; ++kk) {
      const double q = k.prim[(kk * 5 + 0) * k.stride + j];
      const double Q[3] = {k.prim[(kk * 5 + 1) * k.stride + j], k.prim[(kk * 5 + 2) * k.stride + j], k.prim[(kk * 5 + 3) * k.stride + j]};
      const double Kcd = k.prim[(kk * 5 + 4) * k.stride + j];
      const double pq = p + q, rpq = 1.0 / pq, rho = p * q * rpq;
      const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
      const double x = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
      const double pref = Kab * Kcd * sqrt(rpq);
      rys_roots_rt(N, x, w.rys, u, wt);
      const bool swb = swap_centre(P, g.A, g.AB), swk = swap_centre(Q, g.C, g.CD);
      for (int r = 0; r < N; ++r) {
        const double t2 = u[r];
        const double b00 = 0.5 * t2 * rpq;
        const double b10 = (1.0 - q * t2 * rpq) * 0.5 / p;
        const double b01 = (1.0 - p * t2 * rpq) * 0.5 / q;
        double* G[3] = {gx, gy, gz};
        for (int ax = 0; ax < 3; ++ax) {
          const double c00 = (P[ax] - g.A[ax]) + (swb ? g.AB[ax] : 0.0) - q * t2 * rpq * PQ[ax];
          const double c00p = (Q[ax] - g.C[ax]) + (swk ? g.CD[ax] : 0.0) + p * t2 * rpq * PQ[ax];
          fill_2d<LC>(G[ax], na, nb, nc, nd, ax == 2 ? pref * wt[r] : 1.0, c00, c00p, b10, b01, b00, g.AB[ax], g.CD[ax], swb, swk);
        }
        cons(gx, gy, gz);
      }
    }
  }
}

// ---- consumers ------------------------------------------------------------------------------------------------
// Cartesian components in the order lx descending, then ly descending.
#define FOR_CART(l, cx, cy, cz, idx) \
  for (int cx = (l), idx = 0; cx >= 0; --cx) for (int cy = (l) - cx, cz = 0; cy >= 0; --cy, ++idx, cz = (l) - cx - cy)

struct DigestConsumer {   // six updates of Alg. 2 lines 8-13, before contraction
  const double* D; double* J; double* K; int n; int a0, b0, c0, d0; int la, lb, lc, ld; double f;
  __device__ void operator()(const double* gx, const double* gy, const double* gz) {
    const int nb = lb + 1, nc = lc + 1, nd = ld + 1;
    for (int ax = la, ia = 0; ax >= 0; --ax) for (int ay = la - ax; ay >= 0; --ay, ++ia) { const int az = la - ax - ay;
    for (int bx = lb, ib = 0; bx >= 0; --bx) for (int by = lb - bx; by >= 0; --by, ++ib) { const int bz = lb - bx - by;
    for (int cx = lc, ic = 0; cx >= 0; --cx) for (int cy = lc - cx; cy >= 0; --cy, ++ic) { const int cz = lc - cx - cy;
    for (int dx = ld, id = 0; dx >= 0; --dx) for (int dy = ld - dx; dy >= 0; --dy, ++id) { const int dz = ld - dx - dy;
      const double v = f * gx[((ax * nb + bx) * nc + cx) * nd + dx] * gy[((ay * nb + by) * nc + cy) * nd + dy] *
                       gz[((az * nb + bz) * nc + cz) * nd + dz];
      const long a = a0 + ia, b = b0 + ib, c = c0 + ic, d = d0 + id;
      atomic_add(J + a * n + b, v * D[c * n + d]);
      atomic_add(J + c * n + d, v * D[a * n + b]);
      atomic_add(K + a * n + c, v * D[b * n + d]);
      atomic_add(K + b * n + d, v * D[a * n + c]);
      atomic_add(K + a * n + d, v * D[b * n + c]);
      atomic_add(K + b * n + c, v * D[a * n + d]);
    }}}}
  }
};

struct StoreConsumer {    // accumulate the Cartesian block [nca][ncb][ncc][ncd] (element e at out[e * stride]); one thread owns the block
  double* out; int la, lb, lc, ld; long stride;
  __device__ void operator()(const double* gx, const double* gy, const double* gz) {
    const int nb = lb + 1, nc = lc + 1, nd = ld + 1;
    long e = 0;
    for (int ax = la; ax >= 0; --ax) for (int ay = la - ax; ay >= 0; --ay) { const int az = la - ax - ay;
    for (int bx = lb; bx >= 0; --bx) for (int by = lb - bx; by >= 0; --by) { const int bz = lb - bx - by;
    for (int cx = lc; cx >= 0; --cx) for (int cy = lc - cx; cy >= 0; --cy) { const int cz = lc - cx - cy;
    for (int dx = ld; dx >= 0; --dx) for (int dy = ld - dx; dy >= 0; --dy, ++e) { const int dz = ld - dx - dy;
      out[e * stride] += gx[((ax * nb + bx) * nc + cx) * nd + dx] * gy[((ay * nb + by) * nc + cy) * nd + dy] *
                         gz[((az * nb + bz) * nc + cz) * nd + dz];
    }}}}
  }
};

template <int LC>
__global__ void __launch_bounds__(128) generic_jk_kernel(Work w) {
  int i, j; double f;
  if (!locate(w, i, j, f)) return;
  QuartetGeom g; load_geom(w, i, j, g);
  DigestConsumer c{w.D, w.J, w.K, w.nao, w.bra.ao[i].x, w.bra.ao[i].y, w.ket.ao[j].x, w.ket.ao[j].y, g.la, g.lb, g.lc, g.ld, f};
  quartet_loop<LC>(w, i, j, g, c);
}

// list mode only: element e of block t of Cartesian integrals is accumulated at out[off[t] + e * stride] (zeroed by the caller).
// stride 1: one contiguous block per quartet; off[t] = t, stride = number of items: element-major, so that the read-modify-write
// of the 32 threads of a warp coalesces (the Schwarz pass of plan creation)
template <int LC>
__global__ void __launch_bounds__(128) generic_store_kernel(Work w, double* out, const long long* off, long stride) {
  int i, j; double f;
  if (!locate(w, i, j, f)) return;
  const long t = (long)(blockIdx.x * w.nshard + w.shard) * (blockDim.x * blockDim.y) + threadIdx.y * blockDim.x + threadIdx.x;
  QuartetGeom g; load_geom(w, i, j, g);
  StoreConsumer c{out + off[t], g.la, g.lb, g.lc, g.ld, stride};
  if (w.kb_split > 1) quartet_loop<LC>(w, i, j, g, c, (int)(t / w.kb_items), w.kb_split);   // a share of the bra primitive pairs
  else quartet_loop<LC>(w, i, j, g, c);
}

// ---- gradient (Algorithm 4; Eq. 11) -------------------------------------------
// 2-D integrals raised by one on a, b and c; F_a[I](i..) = 2 alpha_a I(i+1,j,k,l) - i I(i-1,j,k,l) on the differentiated
// centre and axis; the fourth centre follows from translational invariance.  Per unique quartet
//   PJ = 4 f D_ab D_cd,  PK = 2 f (D_ac D_bd + D_ad D_bc)
// and 18 accumulators (3 centres x 3 axes x {J,K}); 24 atomics at the end ("12 atomics per quartet").
template <int LC>
__global__ void __launch_bounds__(128) generic_grad_kernel(Work w) {
  int i, j; double f;
  if (!locate(w, i, j, f)) return;
  QuartetGeom g; load_geom(w, i, j, g);
  const PairSet& b = w.bra; const PairSet& k = w.ket;
  const int la = g.la, lb = g.lb, lc = g.lc, ld = g.ld;
  const int N = nroots_of(la + lb + lc + ld + 1);
  const int na = la + 2, nb = lb + 2, nc = lc + 2, nd = ld + 1;
  const int a0 = b.ao[i].x, b0 = b.ao[i].y, c0 = k.ao[j].x, d0 = k.ao[j].y;
  const int n = w.nao;
  const double* D = w.D;
  double gx[Cap<LC>::G1], gy[Cap<LC>::G1], gz[Cap<LC>::G1];
  double u[Cap<LC>::NR], wt[Cap<LC>::NR];
  double accJ[9], accK[9];
  for (int x = 0; x < 9; ++x) accJ[x] = accK[x] = 0.0;
  const int Ka = b.npp, Kc = k.npp;
  for (int kb = 0; kb < Ka; ++kb) {
    const double p = b.prim[(kb * 5 + 0) * b.stride + i];
    const double P[3] = {b.prim[(kb * 5 + 1) * b.stride + i], b.prim[(kb * 5 + 2) * b.stride + i], b.prim[(kb * 5 + 3) * b.stride + i]};
    const double Kab = b.prim[(kb * 5 + 4) * b.stride + i];
    const double ea2 = 2.0 * b.aexp[(kb * 2 + 0) * b.stride + i], eb2 = 2.0 * b.aexp[(kb * 2 + 1) * b.stride + i];
    for (int kk = 0; kk < Kc; ++kk) {
      const double q = k.prim[(kk * 5 + 0) * k.stride + j];
      const double Q[3] = {k.prim[(kk * 5 + 1) * k.stride + j], k.prim[(kk * 5 + 2) * k.stride + j], k.prim[(kk * 5 + 3) * k.stride + j]};
      const double Kcd = k.prim[(kk * 5 + 4) * k.stride + j];
      const double ec2 = 2.0 * k.aexp[(kk * 2 + 0) * k.stride + j];
      const double pq = p + q, rpq = 1.0 / pq, rho = p * q * rpq;
      const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
      const double x = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
      const double pref = Kab * Kcd * sqrt(rpq);
      rys_roots_rt(N, x, w.rys, u, wt);
      const bool swb = swap_centre(P, g.A, g.AB), swk = swap_centre(Q, g.C, g.CD);
      for (int r = 0; r < N; ++r) {
        const double t2 = u[r];
        const double b00 = 0.5 * t2 * rpq;
        const double b10 = (1.0 - q * t2 * rpq) * 0.5 / p;
        const double b01 = (1.0 - p * t2 * rpq) * 0.5 / q;
        double* G[3] = {gx, gy, gz};
        for (int ax = 0; ax < 3; ++ax) {
          const double c00 = (P[ax] - g.A[ax]) + (swb ? g.AB[ax] : 0.0) - q * t2 * rpq * PQ[ax];
          const double c00p = (Q[ax] - g.C[ax]) + (swk ? g.CD[ax] : 0.0) + p * t2 * rpq * PQ[ax];
          fill_2d<LC>(G[ax], na, nb, nc, nd, ax == 2 ? pref * wt[r] : 1.0, c00, c00p, b10, b01, b00, g.AB[ax], g.CD[ax], swb, swk);
        }
        const int sa = nb * nc * nd, sb = nc * nd, sc = nd;
        for (int axx = la, ia = 0; axx >= 0; --axx) for (int ay = la - axx; ay >= 0; --ay, ++ia) { const int az = la - axx - ay;
        for (int bx = lb, ib = 0; bx >= 0; --bx) for (int by = lb - bx; by >= 0; --by, ++ib) { const int bz = lb - bx - by;
        for (int cx = lc, ic = 0; cx >= 0; --cx) for (int cy = lc - cx; cy >= 0; --cy, ++ic) { const int cz = lc - cx - cy;
        for (int dx = ld, id = 0; dx >= 0; --dx) for (int dy = ld - dx; dy >= 0; --dy, ++id) { const int dz = ld - dx - dy;
          const long a = a0 + ia, bb = b0 + ib, c = c0 + ic, d = d0 + id;
          const double PJ = 4.0 * f * D[a * n + bb] * D[c * n + d];
          const double PK = 2.0 * f * (D[a * n + c] * D[bb * n + d] + D[a * n + d] * D[bb * n + c]);
          const int pw[3][4] = {{axx, bx, cx, dx}, {ay, by, cy, dy}, {az, bz, cz, dz}};
          double val[3], dA[3], dB[3], dC[3];
          for (int ax = 0; ax < 3; ++ax) {
            const double* Gx = G[ax];
            const int e = pw[ax][0] * sa + pw[ax][1] * sb + pw[ax][2] * sc + pw[ax][3];
            val[ax] = Gx[e];
            dA[ax] = ea2 * Gx[e + sa] - (pw[ax][0] > 0 ? pw[ax][0] * Gx[e - sa] : 0.0);
            dB[ax] = eb2 * Gx[e + sb] - (pw[ax][1] > 0 ? pw[ax][1] * Gx[e - sb] : 0.0);
            dC[ax] = ec2 * Gx[e + sc] - (pw[ax][2] > 0 ? pw[ax][2] * Gx[e - sc] : 0.0);
          }
          const double oth[3] = {val[1] * val[2], val[0] * val[2], val[0] * val[1]};
          for (int ax = 0; ax < 3; ++ax) {
            const double ga = dA[ax] * oth[ax], gb = dB[ax] * oth[ax], gc = dC[ax] * oth[ax];
            accJ[ax] += PJ * ga; accJ[3 + ax] += PJ * gb; accJ[6 + ax] += PJ * gc;
            accK[ax] += PK * ga; accK[3 + ax] += PK * gb; accK[6 + ax] += PK * gc;
          }
        }}}}
      }
    }
  }
  const int atA = b.atom[i].x, atB = b.atom[i].y, atC = k.atom[j].x, atD = k.atom[j].y;
  for (int ax = 0; ax < 3; ++ax) {
    atomic_add(w.gJ + 3 * atA + ax, accJ[ax]);     atomic_add(w.gK + 3 * atA + ax, accK[ax]);
    atomic_add(w.gJ + 3 * atB + ax, accJ[3 + ax]); atomic_add(w.gK + 3 * atB + ax, accK[3 + ax]);
    atomic_add(w.gJ + 3 * atC + ax, accJ[6 + ax]); atomic_add(w.gK + 3 * atC + ax, accK[6 + ax]);
    atomic_add(w.gJ + 3 * atD + ax, -(accJ[ax] + accJ[3 + ax] + accJ[6 + ax]));
    atomic_add(w.gK + 3 * atD + ax, -(accK[ax] + accK[3 + ax] + accK[6 + ax]));
  }
}

}  // namespace

static bool needs_hi(const Work& w) { return w.bra.la > 4 || w.bra.lb > 4 || w.ket.la > 4 || w.ket.lb > 4; }   // any h or i shell

static int grid_of(const Work& w, int threads, int total_blocks_dense) {
  const int total = w.list ? (w.nlist + threads - 1) / threads : total_blocks_dense;
  return (total + w.nshard - 1) / w.nshard;
}

cudaError_t launch_generic_jk(const Work& w, int nblocks_dense, cudaStream_t s) {
  dim3 block(GENERIC_BJ, GENERIC_BI);
  const int grid = grid_of(w, GENERIC_BJ * GENERIC_BI, nblocks_dense);
  if (grid <= 0) return cudaSuccess;
  if (needs_hi(w)) generic_jk_kernel<6><<<grid, block, 0, s>>>(w); else generic_jk_kernel<4><<<grid, block, 0, s>>>(w);
  return cudaGetLastError();
}

cudaError_t launch_generic_store(const Work& w, double* out, const long long* off, long stride, cudaStream_t s) {
  dim3 block(GENERIC_BJ, GENERIC_BI);
  const int grid = grid_of(w, GENERIC_BJ * GENERIC_BI, 0);
  if (grid <= 0) return cudaSuccess;
  if (needs_hi(w)) generic_store_kernel<6><<<grid, block, 0, s>>>(w, out, off, stride); else generic_store_kernel<4><<<grid, block, 0, s>>>(w, out, off, stride);
  return cudaGetLastError();
}

cudaError_t launch_generic_grad(const Work& w, int nblocks_dense, cudaStream_t s) {
  dim3 block(GENERIC_GRAD_BJ, GENERIC_GRAD_BI);
  const int grid = grid_of(w, GENERIC_GRAD_BJ * GENERIC_GRAD_BI, nblocks_dense);
  if (grid <= 0) return cudaSuccess;
  if (needs_hi(w)) generic_grad_kernel<6><<<grid, block, 0, s>>>(w); else generic_grad_kernel<4><<<grid, block, 0, s>>>(w);
  return cudaGetLastError();
}

}  // namespace eri
