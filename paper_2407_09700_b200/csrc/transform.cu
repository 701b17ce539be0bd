// transform.cu -- matrix-level Cartesian <-> real-solid-harmonic transforms (DESIGN.md step S5/S7), spherical
// blocks for the diagnostic entry points, the Schwarz reduction (Eq. 7), and two small diagnostics.
// The kernels digest in the Cartesian AO basis: D_cart = T^T D T once per call, J = T (2 (Jt + Jt^T)) T^T and
// K = T (Kt + Kt^T) T^T at the end (reading R9) -- the paper never states how spherical functions are handled.
#include <mutex>

#include "../../include/eri.h"
#include "eri_dev.cuh"
#include "launch.h"

namespace eri {
namespace {

__host__ __device__ constexpr int c2s_off(int l) { int off = 0; for (int k = 0; k < l; ++k) off += nsph(k) * ncart(k); return off; }
constexpr int C2S_SIZE = c2s_off(LMAX + 1);   // 840 doubles for l <= 6
__constant__ double c_c2s[C2S_SIZE];          // l-th table at c2s_off(l), ns(l) x nc(l) row-major

__global__ void sph2cart_kernel(ShellMap m, const double* __restrict__ Ds, double* __restrict__ Dc) {
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  const long n2 = (long)m.nao_cart * m.nao_cart;
  if (t >= n2) return;
  const int p = (int)(t / m.nao_cart), q = (int)(t % m.nao_cart);
  const int sp = m.cart2sh[p], sq = m.cart2sh[q];
  const int lp = m.sh_l[sp], lq = m.sh_l[sq];
  const int cp = p - m.sh_cart[sp], cq = q - m.sh_cart[sq];
  const double* Tp = c_c2s + c2s_off(lp); const double* Tq = c_c2s + c2s_off(lq);
  const int ncp = ncart(lp), ncq = ncart(lq);
  const int p0 = m.sh_sph[sp], q0 = m.sh_sph[sq];
  double acc = 0.0;
  for (int a = 0; a < nsph(lp); ++a) {
    const double ta = Tp[a * ncp + cp];
    if (ta == 0.0) continue;
    double row = 0.0;
    for (int b = 0; b < nsph(lq); ++b) row += Ds[(long)(p0 + a) * m.nao + q0 + b] * Tq[b * ncq + cq];
    acc += ta * row;
  }
  Dc[t] = acc;
}

__global__ void cart2sph_kernel(ShellMap m, const double* __restrict__ Mc, double* __restrict__ Ms, double alpha, int sym) {
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  const long n2 = (long)m.nao * m.nao;
  if (t >= n2) return;
  const int p = (int)(t / m.nao), q = (int)(t % m.nao);
  const int sp = m.sph2sh[p], sq = m.sph2sh[q];
  const int lp = m.sh_l[sp], lq = m.sh_l[sq];
  const int a = p - m.sh_sph[sp], b = q - m.sh_sph[sq];
  const int ncp = ncart(lp), ncq = ncart(lq);
  const double* Tp = c_c2s + c2s_off(lp) + a * ncp; const double* Tq = c_c2s + c2s_off(lq) + b * ncq;
  const int p0 = m.sh_cart[sp], q0 = m.sh_cart[sq];
  const long n = m.nao_cart;
  double acc = 0.0;
  for (int cp = 0; cp < ncp; ++cp) {
    if (Tp[cp] == 0.0) continue;
    double row = 0.0;
    for (int cq = 0; cq < ncq; ++cq) {
      double v = Mc[(p0 + cp) * n + q0 + cq];
      if (sym) v += Mc[(q0 + cq) * n + p0 + cp];
      row += v * Tq[cq];
    }
    acc += Tp[cp] * row;
  }
  Ms[t] = alpha * acc;
}

// one block per quartet; four quarter transforms through shared memory would be faster, but this is a diagnostic path:
// each thread forms one spherical element by the plain four-fold sum, skipping zero coefficients.
__global__ void block_c2s_kernel(ShellMap m, const int* __restrict__ q4, const double* __restrict__ cart,
                                 const long long* __restrict__ coff, double* __restrict__ out, const long long* __restrict__ ooff) {
  const int t = blockIdx.x;
  int l[4], nc[4], ns[4];
  for (int x = 0; x < 4; ++x) { l[x] = m.sh_l[q4[4 * t + x]]; nc[x] = ncart(l[x]); ns[x] = nsph(l[x]); }
  const double* src = cart + coff[t];
  double* dst = out + ooff[t];
  const int ntot = ns[0] * ns[1] * ns[2] * ns[3];
  for (int e = threadIdx.x; e < ntot; e += blockDim.x) {
    int r = e;
    const int d = r % ns[3]; r /= ns[3];
    const int c = r % ns[2]; r /= ns[2];
    const int b = r % ns[1]; const int a = r / ns[1];
    const double* Ta = c_c2s + c2s_off(l[0]) + a * nc[0];
    const double* Tb = c_c2s + c2s_off(l[1]) + b * nc[1];
    const double* Tc = c_c2s + c2s_off(l[2]) + c * nc[2];
    const double* Td = c_c2s + c2s_off(l[3]) + d * nc[3];
    double acc = 0.0;
    for (int ia = 0; ia < nc[0]; ++ia) { if (Ta[ia] == 0.0) continue;
      double sb = 0.0;
      for (int ib = 0; ib < nc[1]; ++ib) { if (Tb[ib] == 0.0) continue;
        double sc = 0.0;
        for (int ic = 0; ic < nc[2]; ++ic) { if (Tc[ic] == 0.0) continue;
          double sd = 0.0;
          const double* row = src + (((long)ia * nc[1] + ib) * nc[2] + ic) * nc[3];
          for (int id = 0; id < nc[3]; ++id) sd += Td[id] * row[id];
          sc += Tc[ic] * sd;
        }
        sb += Tb[ib] * sc;
      }
      acc += Ta[ia] * sb;
    }
    dst[e] = acc;
  }
}

// one warp per pair: spherical diagonal (st|st) from the Cartesian block M[(ab),(a'b')]
__global__ void schwarz_diag_kernel(int la, int lb, int n, long stride, const double* __restrict__ cart, double* __restrict__ Q) {
  const int t = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
  const int lane = threadIdx.x % 32;
  if (t >= n) return;
  const int nca = ncart(la), ncb = ncart(lb), nab = nca * ncb;
  const double* M = cart + t;   // element-major: element e of this pair at M[e * stride]
  const double* Ta = c_c2s + c2s_off(la); const double* Tb = c_c2s + c2s_off(lb);
  double best = 0.0;
  for (int st = lane; st < nsph(la) * nsph(lb); st += 32) {
    const int s = st / nsph(lb), tt = st % nsph(lb);
    double acc = 0.0;
    for (int a = 0; a < nca; ++a) { const double ta = Ta[s * nca + a]; if (ta == 0.0) continue;
      for (int b = 0; b < ncb; ++b) { const double tb = Tb[tt * ncb + b]; if (tb == 0.0) continue;
        double inner = 0.0;
        const double* row = M + (long)(a * ncb + b) * nab * stride;
        for (int a2 = 0; a2 < nca; ++a2) { const double ta2 = Ta[s * nca + a2]; if (ta2 == 0.0) continue;
          for (int b2 = 0; b2 < ncb; ++b2) inner += ta2 * Tb[tt * ncb + b2] * row[(long)(a2 * ncb + b2) * stride];
        }
        acc += ta * tb * inner;
      }
    }
    best = fmax(best, fabs(acc));
  }
  for (int o = 16; o > 0; o >>= 1) best = fmax(best, __shfl_xor_sync(0xffffffffu, best, o));
  if (lane == 0) Q[t] = sqrt(best);
}

__global__ void rys_diag_kernel(int N, const double* __restrict__ rys, const double* __restrict__ x, int n,
                                double* __restrict__ u, double* __restrict__ w) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  double uu[RYS_NROOTS_MAX], ww[RYS_NROOTS_MAX];
  rys_roots_rt(N, x[t], rys, uu, ww);
  for (int k = 0; k < N; ++k) { u[(long)t * N + k] = uu[k]; w[(long)t * N + k] = ww[k]; }
}

// N <= RYS2_NMAX: the same points through the shared-memory copy of the table (rys_roots_smem, used by the thread-per-quartet
// families); the two routes share coefficients and summation order, so any bit of difference is reported as NaN
template <int N>
__global__ void rys_diag_smem_kernel(const double* __restrict__ rys, const double* __restrict__ x, int n,
                                     double* __restrict__ u, double* __restrict__ w) {
  extern __shared__ __align__(16) double tab[];
  rys_stage_table<N>(tab, rys, threadIdx.x, blockDim.x);
  __syncthreads();
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  double uu[N], ww[N], u2[RYS_NROOTS_MAX], w2[RYS_NROOTS_MAX];
  rys_roots_smem<N>(x[t], tab, rys, uu, ww);
  rys_roots_rt(N, x[t], rys, u2, w2);
  const double bad = __longlong_as_double(0x7ff8000000000000LL);
  for (int k = 0; k < N; ++k) { u[(long)t * N + k] = uu[k] == u2[k] ? uu[k] : bad; w[(long)t * N + k] = ww[k] == w2[k] ? ww[k] : bad; }
}

// ---- density-weighted screening (Eq. 8-9) -------------------------------------------------------------
// P_{a|b} = max |D| over the sub-block of the (spherical) density between shell groups a and b: one pass over D.
__global__ void group_max_kernel(const double* __restrict__ D, int nao, const int* __restrict__ ao_group, int ng,
                                 unsigned long long* __restrict__ pmax) {
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long)nao * nao) return;
  const int i = (int)(t / nao), j = (int)(t - (long)i * nao);
  const double v = fabs(D[t]);
  if (v > 0.0) atomicMax(pmax + ao_group[i] * ng + ao_group[j], (unsigned long long)__double_as_longlong(v));   // non-negative doubles order like integers
}

// ---- allocation-free variant (eri_density_group_max_noalloc, eri.h) ------------------------------------------------------
// The accumulators of the pass over D live in this file-scope array instead of a cudaMalloc'd buffer: every device that loads
// the library holds ERI_NOALLOC_MAX_GROUPS^2 words (32 KB) until the process exits.  In HOST code the name below is a stand-in,
// not a device address: the launcher takes the address once per device with cudaGetSymbolAddress (that device current) and
// passes the pointer to the kernels.  All calls share the array and it keeps the last call's contents.
static __device__ __align__(256) unsigned long long d_group_max_scratch[ERI_NOALLOC_MAX_GROUPS * ERI_NOALLOC_MAX_GROUPS];

// same pass as group_max_kernel, accumulators in `scratch` (zeroed by the launcher); group ids outside 0..ng-1 are ignored
__global__ void group_max_noalloc_kernel(const double* __restrict__ D, int nao, const int* __restrict__ ao_group, int ng,
                                         unsigned long long* __restrict__ scratch) {
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long)nao * nao) return;
  const int i = (int)(t / nao), j = (int)(t - (long)i * nao);
  const int gi = ao_group[i], gj = ao_group[j];
  const double v = fabs(D[t]);
  if (v > 0.0 && (unsigned)gi < (unsigned)ng && (unsigned)gj < (unsigned)ng)
    atomicMax(scratch + gi * ng + gj, (unsigned long long)__double_as_longlong(v));
}

__global__ void group_max_export_kernel(const unsigned long long* __restrict__ scratch, int n, double* __restrict__ P) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n) P[t] = __longlong_as_double((long long)scratch[t]);
}

// per unit u: thr_eff[u] = tau / P_{ab|cd}, P = the largest of the six group sub-block maxima (Eq. 9); per bra pair i the
// kept kets are the prefix of the Schwarz-sorted ket set with q_i q_j >= thr_eff (Alg. 1 lines 12-16 in the limit of fine
// bins), never more than the plan's Schwarz-only count; kept[u] = number of quartets of the unit that pass.
__global__ void dscreen_kernel(const DscreenUnit* __restrict__ units, const unsigned long long* __restrict__ pmax, int ng, double tau,
                               double* __restrict__ thr_eff, unsigned long long* __restrict__ kept) {
  const DscreenUnit U = units[blockIdx.y];
  const int g[4] = {U.g[0], U.g[1], U.g[2], U.g[3]};
  double P = 0.0;
#pragma unroll
  for (int x = 0; x < 4; ++x)
#pragma unroll
    for (int y = 0; y < 4; ++y)
      if (x != y) P = fmax(P, __longlong_as_double((long long)pmax[g[x] * ng + g[y]]));
  const double te = P > 0.0 ? tau / P : 1.0e300;
  if (blockIdx.x == 0 && threadIdx.x == 0) thr_eff[blockIdx.y] = te;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  int cnt = 0;
  if (i < U.nbra) {
    const double qi = U.qb[i];
    int lo = 0, hi = U.count[i];                 // largest prefix with q_i q_j >= thr_eff (q sorted descending)
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (qi * U.qk[mid] >= te) lo = mid + 1; else hi = mid; }
    cnt = lo;
    U.count_dyn[i] = cnt;
  }
  unsigned long long c = cnt;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
  if ((threadIdx.x & 31) == 0 && c) atomicAdd(kept + blockIdx.y, c);
}

// work list of the Schwarz pass: item t is the quartet (pair start+t | pair start+t), its Cartesian block element-major at offset t
// (split > 1: the m quartets split times over, copy s at t = s m + k; the partial blocks are folded by fold_partials_kernel)
__global__ void diag_list_kernel(int2* __restrict__ list, long long* __restrict__ off, int start, int m, int split) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < m * split) { const int k = t % m; list[t] = make_int2(start + k, start + k); off[t] = t; }
}

// cart[e * m * split + k] += the same element of the copies s = 1 .. split - 1 (at + s m)
__global__ void fold_partials_kernel(double* __restrict__ cart, long nelem, int m, int split) {
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= nelem * m) return;
  const long e = idx / m; const int k = (int)(idx - e * m);
  double* p = cart + e * (long)m * split + k;
  double sum = p[0];
  for (int s = 1; s < split; ++s) sum += p[(long)s * m];
  p[0] = sum;
}

// Primitive-pair records of a pair set (eri_dev.cuh "Pair set") computed on the device from the shell data: thread (pair i,
// primitive pair k) writes p, P, K_ab and the two exponents; k = 0 also writes the pair's geometry, AO offsets and atoms.
// Same formulas as upload_pair_class (api.cu), which serves the list plans from the host.
__global__ void build_pairs_kernel(const eri_shell_t* __restrict__ sh, const eri_prim_t* __restrict__ pr, const double* __restrict__ xyz,
                                   const int* __restrict__ cart_off, const int* __restrict__ sa, const int* __restrict__ sb, int n, int Kb, int npp,
                                   long st, double kfac, double* __restrict__ prim, double* __restrict__ geom, double* __restrict__ aexp,
                                   int2* __restrict__ ao, int2* __restrict__ atom) {
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long)n * npp) return;
  const int k = (int)(t / n), i = (int)(t - (long)k * n);
  const eri_shell_t A = sh[sa[i]], B = sh[sb[i]];
  const double RA[3] = {xyz[3 * A.atom], xyz[3 * A.atom + 1], xyz[3 * A.atom + 2]};
  const double RB[3] = {xyz[3 * B.atom], xyz[3 * B.atom + 1], xyz[3 * B.atom + 2]};
  const double ab[3] = {RA[0] - RB[0], RA[1] - RB[1], RA[2] - RB[2]};
  const double r2 = ab[0] * ab[0] + ab[1] * ab[1] + ab[2] * ab[2];
  const int ka = k / Kb, kb = k - ka * Kb;
  const eri_prim_t pa = pr[A.prim_off + ka], pb = pr[B.prim_off + kb];
  const double p = pa.exp + pb.exp;
  prim[((long)k * 5 + 0) * st + i] = p;
#pragma unroll
  for (int x = 0; x < 3; ++x) prim[((long)k * 5 + 1 + x) * st + i] = (pa.exp * RA[x] + pb.exp * RB[x]) / p;
  prim[((long)k * 5 + 4) * st + i] = kfac / p * pa.coef * pb.coef * exp(-pa.exp * pb.exp / p * r2);
  aexp[((long)k * 2 + 0) * st + i] = pa.exp; aexp[((long)k * 2 + 1) * st + i] = pb.exp;
  if (k == 0) {
#pragma unroll
    for (int x = 0; x < 3; ++x) { geom[x * st + i] = RA[x]; geom[(3 + x) * st + i] = ab[x]; }
    geom[6 * st + i] = sa[i] == sb[i] ? 0.5 : 1.0;
    ao[i] = make_int2(cart_off[sa[i]], cart_off[sb[i]]);
    atom[i] = make_int2(A.atom, B.atom);
  }
}

// pair records of a reordered subset of a pair set (plan creation: the Schwarz-sorted kept set and its grouped twin are
// gathered on the device from the set that the Schwarz pass used, instead of being rebuilt on the host and uploaded again)
__global__ void gather_rows_kernel(const double* __restrict__ src, double* __restrict__ dst, const int* __restrict__ idx, int n, int rows,
                                   long sstride, long dstride) {
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long)rows * n) return;
  const int r = (int)(t / n), i = (int)(t - (long)r * n);
  dst[r * dstride + i] = src[r * sstride + idx[i]];
}
__global__ void gather_int2_kernel(const int2* __restrict__ src, int2* __restrict__ dst, const int* __restrict__ idx, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = src[idx[i]];
}

// 16 independent FMA chains per thread; 2 flops per FMA
__global__ void __launch_bounds__(256) fp64_peak_kernel(double* sink, int iters) {
  double a[16];
  const double x = 1.0 + 1e-9 * threadIdx.x, y = 1e-9 * blockIdx.x;
#pragma unroll
  for (int k = 0; k < 16; ++k) a[k] = k * 0.125 + threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 16; ++k) a[k] = fma(a[k], x, y);
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += a[k];
  if (s == 123.456) sink[0] = s;   // never true; keeps the loop alive
}

}  // namespace

cudaError_t upload_c2s(const double* tables) { return cudaMemcpyToSymbol(c_c2s, tables, sizeof(double) * C2S_SIZE); }

cudaError_t launch_sph2cart(const ShellMap& m, const double* Ds, double* Dc, cudaStream_t s) {
  const long n2 = (long)m.nao_cart * m.nao_cart;
  if (n2 == 0) return cudaSuccess;
  sph2cart_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, s>>>(m, Ds, Dc);
  return cudaGetLastError();
}

cudaError_t launch_cart2sph(const ShellMap& m, const double* Mc, double* Ms, double alpha, int sym, cudaStream_t s) {
  const long n2 = (long)m.nao * m.nao;
  if (n2 == 0) return cudaSuccess;
  cart2sph_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, s>>>(m, Mc, Ms, alpha, sym);
  return cudaGetLastError();
}

cudaError_t launch_block_c2s(const ShellMap& m, const int* q4, int n, const double* cart, const long long* coff,
                             double* out, const long long* ooff, cudaStream_t s) {
  if (n <= 0) return cudaSuccess;
  block_c2s_kernel<<<n, 128, 0, s>>>(m, q4, cart, coff, out, ooff);
  return cudaGetLastError();
}

cudaError_t launch_schwarz_diag(int la, int lb, int n, long stride, const double* cart, double* Q, cudaStream_t s) {
  if (n <= 0) return cudaSuccess;
  schwarz_diag_kernel<<<(n + 3) / 4, 128, 0, s>>>(la, lb, n, stride, cart, Q);
  return cudaGetLastError();
}

cudaError_t launch_fold_partials(double* cart, long nelem, int m, int split, cudaStream_t s) {
  if (split <= 1 || m <= 0) return cudaSuccess;
  const long tot = nelem * m;
  fold_partials_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(cart, nelem, m, split);
  return cudaGetLastError();
}

cudaError_t launch_rys_diag(int N, const double* rys, const double* x, int n, double* u, double* w, cudaStream_t s) {
  if (n <= 0) return cudaSuccess;
  const int grid = (n + 127) / 128;
  switch (N) {
#define CASE(NN) case NN: rys_diag_smem_kernel<NN><<<grid, 128, sizeof(double) * rys2_size(NN), s>>>(rys, x, n, u, w); break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6)
#undef CASE
    default: rys_diag_kernel<<<grid, 128, 0, s>>>(N, rys, x, n, u, w);
  }
  static_assert(RYS2_NMAX == 6, "launch_rys_diag lists the second-layout tables up to N = 6");
  return cudaGetLastError();
}

cudaError_t launch_diag_list(int2* list, long long* off, int start, int m, int split, cudaStream_t s) {
  if (m <= 0) return cudaSuccess;
  diag_list_kernel<<<(m * split + 255) / 256, 256, 0, s>>>(list, off, start, m, split);
  return cudaGetLastError();
}

cudaError_t launch_group_max(const double* D, int nao, const int* ao_group, int ng, unsigned long long* pmax, cudaStream_t s) {
  const long n2 = (long)nao * nao;
  if (n2 == 0) return cudaSuccess;
  group_max_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, s>>>(D, nao, ao_group, ng, pmax);
  return cudaGetLastError();
}

// Allocation-free: no cudaMalloc/cudaFree, no allocating library call.  The scratch address is looked up once per device.
cudaError_t launch_group_max_noalloc(const double* D, int nao, const int* ao_group, int ng, double* P, cudaStream_t s) {
  constexpr int MAX_DEVICES = 64;
  static std::mutex mu;
  static unsigned long long* scratch_of[MAX_DEVICES] = {};
  if (ng <= 0) return cudaSuccess;
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
  unsigned long long* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lk(mu);
    if (!scratch_of[dev]) {
      unsigned long long* ptr = nullptr;
      e = cudaGetSymbolAddress((void**)&ptr, d_group_max_scratch);   // this device's copy of the array
      if (e != cudaSuccess) return e;
      scratch_of[dev] = ptr;
    }
    scratch = scratch_of[dev];
  }
  const int n = ng * ng;
  e = cudaMemsetAsync(scratch, 0, sizeof(unsigned long long) * n, s);   // the array keeps the last call's maxima
  if (e != cudaSuccess) return e;
  const long n2 = (long)nao * nao;
  if (n2 > 0) group_max_noalloc_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, s>>>(D, nao, ao_group, ng, scratch);
  group_max_export_kernel<<<(n + 255) / 256, 256, 0, s>>>(scratch, n, P);
  return cudaGetLastError();
}

cudaError_t launch_dscreen(const DscreenUnit* units, int nunits, int max_nbra, const unsigned long long* pmax, int ng, double tau,
                           double* thr_eff, unsigned long long* kept, cudaStream_t s) {
  if (nunits == 0) return cudaSuccess;
  dscreen_kernel<<<dim3((max_nbra + 127) / 128, nunits), 128, 0, s>>>(units, pmax, ng, tau, thr_eff, kept);
  return cudaGetLastError();
}

cudaError_t launch_build_pairs(const eri_shell_t* sh, const eri_prim_t* pr, const double* xyz, const int* cart_off, const int* sa, const int* sb,
                               int n, int Kb, int npp, long st, double kfac, double* prim, double* geom, double* aexp, int2* ao, int2* atom, cudaStream_t s) {
  const long tot = (long)n * npp;
  if (tot <= 0) return cudaSuccess;
  build_pairs_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(sh, pr, xyz, cart_off, sa, sb, n, Kb, npp, st, kfac, prim, geom, aexp, ao, atom);
  return cudaGetLastError();
}

cudaError_t launch_gather_rows(const double* src, double* dst, const int* idx, int n, int rows, long sstride, long dstride, cudaStream_t s) {
  const long tot = (long)rows * n;
  if (tot <= 0) return cudaSuccess;
  gather_rows_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(src, dst, idx, n, rows, sstride, dstride);
  return cudaGetLastError();
}

cudaError_t launch_gather_int2(const int2* src, int2* dst, const int* idx, int n, cudaStream_t s) {
  if (n <= 0) return cudaSuccess;
  gather_int2_kernel<<<(n + 255) / 256, 256, 0, s>>>(src, dst, idx, n);
  return cudaGetLastError();
}

cudaError_t launch_fp64_peak(double* sink, int iters, int blocks, cudaStream_t s) {
  fp64_peak_kernel<<<blocks, 256, 0, s>>>(sink, iters);
  return cudaGetLastError();
}

}  // namespace eri
