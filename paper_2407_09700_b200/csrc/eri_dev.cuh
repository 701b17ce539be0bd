// eri_dev.cuh -- device-side data views and the Rys root/weight routine shared by all kernels of liberi_b200.
// Product code (not test infrastructure); nothing under oracle/ is included, linked or called from here.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace eri {

constexpr int LMAX = 6;   // s..i; tuned kernel families exist up to g, the generic kernels serve h and i
constexpr double PI = 3.14159265358979323846;

__host__ __device__ constexpr int ncart(int l) { return (l + 1) * (l + 2) / 2; }
__host__ __device__ constexpr int nsph(int l) { return 2 * l + 1; }
__host__ __device__ constexpr int nroots_of(int L) { return L / 2 + 1; }  // Eq. 3

// ---------------------------------------------------------------------------------------------------------------
// Rys data buffer (one device allocation, read-only): see api.cu for how it is filled from rys_tables.inc.
//   [0..16)    xmax[N]          switch to the Gauss-Hermite asymptote
//   [16..32)   table offset[N]  (as double)
//   [32..128)  h_n^2 of the 2N-point Gauss-Hermite rule, N-th block at 32 + N(N-1)/2   (N <= 13: 91 values)
//   [128..224) v_n, same indexing
//   [224..)    Chebyshev tables, per N: [interval][k=0..13][2N values]
constexpr int RYS_HDR_XMAX = 0, RYS_HDR_OFF = 16, RYS_HDR_H2 = 32, RYS_HDR_V = 128, RYS_HDR_SIZE = 224;
constexpr int RYS_NROOTS_MAX = 13;   // (ii|ii): floor(24 / 2) + 1; also the gradient of (ii|ih)
__host__ __device__ constexpr double rys_xmax(int N) {
  return N == 1 ? 35.0 : N == 2 ? 45.0 : N == 3 ? 50.0 : 57.5 + 5.0 * (N - 4);   // gen_rys_tables.py XMAX (checked in api.cu)
}
__host__ __device__ constexpr int rys_nint(int N) { return (int)(rys_xmax(N) / 2.5 + 0.5); }
__host__ __device__ constexpr int rys_offset(int N) {  // doubles before the N-th table
  int off = 0;
  for (int n = 1; n < N; ++n) off += rys_nint(n) * 14 * 2 * n;
  return off;
}

// Roots u_n = t_n^2 and weights w_n of the N-point rule for exp(-x t^2) on [0,1] (Eq. 1).
// NN may be a compile-time constant (the loops unroll) or a run-time value.
template <typename Int>
__device__ __forceinline__ void rys_roots_impl(Int NN, int table_off, double xmax, double x,
                                               const double* __restrict__ rys, double* u, double* w) {
  const int N = NN;
  if (x >= xmax) {
    const double rx = 1.0 / x, rs = sqrt(rx);
    const double* h2 = rys + RYS_HDR_H2 + N * (N - 1) / 2;
    const double* v = rys + RYS_HDR_V + N * (N - 1) / 2;
#pragma unroll
    for (int n = 0; n < N; ++n) { u[n] = h2[n] * rx; w[n] = v[n] * rs; }
    return;
  }
  int iv = (int)(x * 0.4);
  const double s = (x - (2.5 * iv + 1.25)) * 0.8, s2 = 2.0 * s;
  const double* c = rys + RYS_HDR_SIZE + table_off + iv * (28 * N);
#pragma unroll
  for (int n = 0; n < 2 * N; ++n) {
    double b1 = c[13 * 2 * N + n], b2 = 0.0;
#pragma unroll
    for (int k = 12; k >= 1; --k) {
      const double t = fma(s2, b1, c[k * 2 * N + n] - b2);
      b2 = b1; b1 = t;
    }
    const double val = fma(s, b1, c[n] - b2);
    if (n < N) u[n] = val; else w[n - N] = val;
  }
}

template <int N>
__device__ __forceinline__ void rys_roots(double x, const double* __restrict__ rys, double* u, double* w) {
  rys_roots_impl<int>(N, rys_offset(N), rys_xmax(N), x, rys, u, w);
}

// ---------------------------------------------------------------------------------------------------------------
// Shared-memory copy of one N's Chebyshev table for the thread-per-quartet families (tile, register, tile gradient).
// There every lane has its own x, hence its own interval: read from global memory, the 28 N coefficient loads of a
// primitive quartet touch up to 32 different 128-byte lines each and the L1/TEX data pipe, not the FP64 pipe, bounds
// the low-l classes (profiles/r02_cfg3.md: 75 % of its peak, 7 sectors per request).  The second layout
//   [interval][value n = 0..2N-1 (u_0.., w_0..)][k = 0..13]
// keeps the 14 coefficients of a value contiguous, so a lane fetches them with seven 128-bit shared loads; lanes in the
// same interval read the same address (broadcast); the interval stride is padded to 2 (mod 16) doubles, i.e. to 1 (mod 8)
// 16-byte slots, so that different intervals fall into different slots of a 128-byte wavefront.
// The buffer holds the layout after the first one, at RYS2_BASE (16-byte aligned).
constexpr int RYS_TABLE_DOUBLES = 83860;                       // = RYS_TABLE_SIZE of rys_tables.inc (checked in api.cu)
constexpr int RYS2_BASE = RYS_HDR_SIZE + RYS_TABLE_DOUBLES;    // even: 16-byte aligned
constexpr int RYS2_NMAX = 6;                                   // classes of the thread-per-quartet families have N <= 6
__host__ __device__ constexpr int rys2_stride(int N) { int s = 28 * N; while (s % 16 != 2) ++s; return s; }
__host__ __device__ constexpr int rys2_size(int N) { return rys_nint(N) * rys2_stride(N); }
__host__ __device__ constexpr int rys2_offset(int N) { int off = 0; for (int n = 1; n < N; ++n) off += rys2_size(n); return off; }

// all threads of the block: copy the class's table to shared memory (dst 16-byte aligned); the caller synchronises
template <int N>
__device__ __forceinline__ void rys_stage_table(double* __restrict__ dst, const double* __restrict__ rys, int tid, int nthreads) {
  static_assert(N <= RYS2_NMAX, "no second-layout table for this N");
  const double2* src = reinterpret_cast<const double2*>(rys + RYS2_BASE + rys2_offset(N));
  double2* d = reinterpret_cast<double2*>(dst);
  for (int i = tid; i < rys2_size(N) / 2; i += nthreads) d[i] = src[i];
}

// same rule, same arithmetic and summation order as rys_roots_impl (bit-identical results), coefficients from `tab`
template <int N>
__device__ __forceinline__ void rys_roots_smem(double x, const double* __restrict__ tab, const double* __restrict__ rys, double* u, double* w) {
  if (x >= rys_xmax(N)) {
    const double rx = 1.0 / x, rs = sqrt(rx);
    const double* h2 = rys + RYS_HDR_H2 + N * (N - 1) / 2;
    const double* v = rys + RYS_HDR_V + N * (N - 1) / 2;
#pragma unroll
    for (int n = 0; n < N; ++n) { u[n] = h2[n] * rx; w[n] = v[n] * rs; }
    return;
  }
  const int iv = (int)(x * 0.4);
  const double s = (x - (2.5 * iv + 1.25)) * 0.8, s2 = 2.0 * s;
  const double2* c = reinterpret_cast<const double2*>(tab + iv * rys2_stride(N));
#pragma unroll
  for (int n = 0; n < 2 * N; ++n) {
    const double2 p6 = c[n * 7 + 6];
    double b1 = p6.y, b2 = 0.0;
    double t = fma(s2, b1, p6.x - b2); b2 = b1; b1 = t;           // k = 12
#pragma unroll
    for (int j = 5; j >= 1; --j) {
      const double2 pj = c[n * 7 + j];
      t = fma(s2, b1, pj.y - b2); b2 = b1; b1 = t;                // k = 2j + 1
      t = fma(s2, b1, pj.x - b2); b2 = b1; b1 = t;                // k = 2j
    }
    const double2 p0 = c[n * 7];
    t = fma(s2, b1, p0.y - b2); b2 = b1; b1 = t;                  // k = 1
    const double val = fma(s, b1, p0.x - b2);
    if (n < N) u[n] = val; else w[n - N] = val;
  }
}
__device__ inline void rys_roots_rt(int N, double x, const double* __restrict__ rys, double* u, double* w) {
  rys_roots_impl<int>(N, (int)rys[RYS_HDR_OFF + N], rys[RYS_HDR_XMAX + N], x, rys, u, w);
}

// ---------------------------------------------------------------------------------------------------------------
// Pair set |ab, KaKb}: all kept shell pairs of one (shell group, shell group) combination, sorted by
// decreasing Schwarz factor.  SoA with the pair index fastest so that one-thread-per-quartet kernels coalesce.
//   prim[(k*5 + f)*stride + i], f: 0 p = alpha+beta, 1..3 P = (alpha A + beta B)/p,
//                               4 Kab = sqrt(2) pi^(5/4) / p * c_a c_b exp(-alpha beta / p |AB|^2)
//   geom[f*stride + i], f: 0..2 A (centre of the first shell), 3..5 A - B, 6 pair weight (1/2 if both shells are the same)
//   aexp[(k*2 + f)*stride + i], f: 0 alpha_a, 1 alpha_b            (gradient only)
//   ao[i]   = (cartesian AO offset of first shell, of second shell);  atom[i] = (atom of first, of second)
struct PairSet {
  const double* prim;
  const double* geom;
  const double* aexp;
  const double* q;   // Schwarz factor per pair, descending
  const int2* ao;
  const int2* atom;
  int npair, stride, npp, la, lb;
};

// One (bra pair set, ket pair set) work unit.
//  dense mode (list == nullptr): bra rows of BI pairs x ket blocks of BJ pairs; quartet (i,j) is evaluated iff
//    j < ket_count[i] (prefix of the Schwarz-sorted ket set, already cut to j <= i when bra set == ket set).
//    Block b belongs to the row r with row_off[r] <= b < row_off[r+1].
//  list mode: work item t is the quartet (list[t].x, list[t].y); weight 1.
struct Work {
  PairSet bra, ket;
  const int* ket_count;
  const int* row_off;
  int nrows;
  int same;          // bra set == ket set: the diagonal quartet (i,i) carries another factor 1/2
  const int2* list;
  int nlist;
  const double* rys;
  const double* D;   // Cartesian-AO density, nao x nao
  double* J;
  double* K;
  double* gJ;        // gradient accumulators, natm*3
  double* gK;
  int nao;
  int shard, nshard; // this process runs the blocks b = blockIdx.x * nshard + shard (eri_plan_set_shard)
  // tile family (tile_kernel.cuh): bra/ket are GROUPED pair sets (chunks of 32 slots sharing the first shell, q < 0 marks
  // a padding slot); row r = the BI bra slots starting at row_slot[r], its blocks = the first row_off[r+1]-row_off[r] ket
  // chunks; a quartet is evaluated iff q_i * q_j >= thr (and j <= i when bra set == ket set) -- the same set as dense mode.
  const int* row_slot;
  double thr;
  int grad_ch;       // cooperative gradient kernel: bra pairs per task (Unit::gBI)
  // density-weighted screening (Eq. 8-9; eri_plan_build_jk_dscreen): the unit's effective threshold
  // tau / P_{ab|cd} in device memory (tile family; the other families get a per-call ket_count); nullptr: use thr
  const double* thr_dev;
  // generic store kernel, Schwarz pass of deeply contracted pair sets (api.cu schwarz_enqueue): the list holds kb_items quartets
  // kb_split times over; copy s = t / kb_items evaluates the bra primitive pairs s, s + kb_split, ... into its own block.  0: whole quartets.
  int kb_split, kb_items;
};

__device__ __forceinline__ void atomic_add(double* p, double v) { atomicAdd(p, v); }

// locate the row of block b: largest r with row_off[r] <= b
__device__ __forceinline__ int find_row(const int* __restrict__ row_off, int nrows, int b) {
  int lo = 0, hi = nrows;  // row_off has nrows+1 entries
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (row_off[mid] <= b) lo = mid; else hi = mid;
  }
  return lo;
}

// the same with the 32 lanes of a warp probing 32 pivots per round (3 rounds of dependent loads instead of 13 for 8192 rows);
// every lane returns the row.  Must be called by all lanes of the warp.
__device__ __forceinline__ int find_row_warp(const int* __restrict__ row_off, int nrows, int b, int lane) {
  int lo = 0, hi = nrows;   // invariant: row_off[lo] <= b < row_off[hi]
  while (hi - lo > 1) {
    const int stride = (hi - lo + 31) >> 5;
    const int idx = lo + lane * stride;
    const bool le = idx < hi && row_off[idx] <= b;
    const int t = __popc(__ballot_sync(0xffffffffu, le));   // lanes 0 .. t-1 are true (row_off is non-decreasing), t >= 1
    lo += (t - 1) * stride;
    hi = min(hi, lo + stride);
  }
  return lo;
}

}  // namespace eri
