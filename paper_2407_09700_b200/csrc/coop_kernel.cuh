// coop_kernel.cuh -- cooperative family of J/K kernels (family W).
// One WARP per shell quartet.  The paper keeps the 2-D integrals of all roots of a quartet in per-thread local memory
// (Algorithm 3) and is bound by local-memory traffic; here the 32 lanes share them
// through shared memory:
//   phase 1  lane (root r, axis x) builds I_x(i,j,k,l; t_r) -- vertical recurrence, then horizontal transfer on both
//            sides at the 2-D level (reading R5), built on the centre nearer to P resp. Q
//            -- and stores it to the warp's shared-memory slab S[axis][root][i][j][k][l];
//   phase 2  lane `ab` owns the Cartesian bra component pair (a,b) (several per lane if nab > 32) and accumulates
//            g[cd] = sum_r X Y Z for every ket component pair in registers (Eq. 1 and Eq. 5): per
//            root 3 (lc+1)(ld+1) shared loads feed 2 nc(lc) nc(ld) FP64 operations;
//   phase 3  contract-then-digest (the six updates of Alg. 2 lines 8-13) straight from registers:
//            J_ab is complete per lane; K partial sums over d resp. c are formed per lane, summed over the lanes
//            that share a resp. b through the (now dead) slab, and leave as one FP64 atomic per block element;
//            J_cd is summed in registers over the bra pairs of the warp's task and reduced across lanes once per task.
// A task is one ket pair and a run of CH consecutive bra pairs of the Schwarz-sorted tile row.
// Large classes give a quartet to TW = 2, 4 or 8 warps (a "group", synchronised with a named barrier) so that the
// accumulators per lane, ceil(nab / 32 TW) * ncd, stay in registers.
#pragma once
#include "eri_dev.cuh"
#include "launch.h"

namespace eri {

constexpr int COOP_WARPS = 4;    // warps (= ket pairs) per block
constexpr int COOP_CH = 16;      // bra pairs per task

// one root of the N-point rule (same tables and asymptote as rys_roots_impl)
template <int N>
__device__ __forceinline__ void rys_root_one(double x, const double* __restrict__ rys, int r, double& u, double& w) {
  if (x >= rys_xmax(N)) {
    const double rx = 1.0 / x;
    u = rys[RYS_HDR_H2 + N * (N - 1) / 2 + r] * rx;
    w = rys[RYS_HDR_V + N * (N - 1) / 2 + r] * sqrt(rx);
    return;
  }
  const int iv = (int)(x * 0.4);
  const double s = (x - (2.5 * iv + 1.25)) * 0.8, s2 = 2.0 * s;
  const double* c = rys + RYS_HDR_SIZE + rys_offset(N) + iv * (28 * N);
  double b1u = c[13 * 2 * N + r], b2u = 0.0, b1w = c[13 * 2 * N + N + r], b2w = 0.0;
#pragma unroll
  for (int k = 12; k >= 1; --k) {
    const double tu = fma(s2, b1u, c[k * 2 * N + r] - b2u), tw = fma(s2, b1w, c[k * 2 * N + N + r] - b2w);
    b2u = b1u; b1u = tu; b2w = b1w; b1w = tw;
  }
  u = fma(s, b1u, c[r] - b2u);
  w = fma(s, b1w, c[N + r] - b2w);
}

// The same root and weight for the lane (root r, axis ax) of a build team whose lanes sit at base + 3 r + ax (phase 1 of the
// paired kernel): the axis-0 lane evaluates the Chebyshev sum of the root, the axis-1 lane that of the weight (the axis-2 lane
// repeats the root's), and the two values are exchanged by shuffles -- half the coefficient loads and FP64 instructions of
// rys_root_one per lane; same arithmetic per value.  `mask`: the lanes of the team (all of them must call).
template <int N>
__device__ __forceinline__ void rys_root_team(double x, const double* __restrict__ rys, int r, int ax, int base, unsigned mask, double& u, double& w) {
  double val;
  const int sel = ax == 1 ? N + r : r;
  if (x >= rys_xmax(N)) {
    const double rx = 1.0 / x;
    val = ax == 1 ? rys[RYS_HDR_V + N * (N - 1) / 2 + r] * sqrt(rx) : rys[RYS_HDR_H2 + N * (N - 1) / 2 + r] * rx;
  } else {
    const int iv = (int)(x * 0.4);
    const double s = (x - (2.5 * iv + 1.25)) * 0.8, s2 = 2.0 * s;
    const double* c = rys + RYS_HDR_SIZE + rys_offset(N) + iv * (28 * N) + sel;
    double b1 = c[13 * 2 * N], b2 = 0.0;
#pragma unroll
    for (int k = 12; k >= 1; --k) {
      const double t = fma(s2, b1, c[k * 2 * N] - b2);
      b2 = b1; b1 = t;
    }
    val = fma(s, b1, c[0] - b2);
  }
  u = __shfl_sync(mask, val, base + 3 * r);
  w = __shfl_sync(mask, val, base + 3 * r + 1);
}

// 2-D integrals of one axis and one root, built on centres 1 (bra) and 3 (ket) and transferred to 2 and 4.
// Element (i1,i2,i3,i4) is stored at dst[i1*s1 + i2*s2 + i3*s3 + i4*s4]; x12 = R1 - R2, x34 = R3 - R4.
template <int L1, int L2, int L3, int L4>
__device__ __forceinline__ void fill_2d_smem(double* __restrict__ dst, int s1, int s2, int s3, int s4, double init, double c00,
                                             double c00p, double b10, double b01, double b00, double x12, double x34) {
  constexpr int NM = L1 + L2, MM = L3 + L4;
  double T[NM + 1][MM + 1];
  T[0][0] = init;
#pragma unroll
  for (int n = 0; n < NM; ++n) T[n + 1][0] = n > 0 ? fma(c00, T[n][0], (n * b10) * T[n - 1][0]) : c00 * T[n][0];
#pragma unroll
  for (int m = 0; m < MM; ++m)
#pragma unroll
    for (int n = 0; n <= NM; ++n) {
      double v = c00p * T[n][m];
      if (m > 0) v = fma(m * b01, T[n][m - 1], v);
      if (n > 0) v = fma(n * b00, T[n - 1][m], v);
      T[n][m + 1] = v;
    }
  // bra transfer in place: after step j, T[i][m] (i <= NM - j) holds I(i, j, m)
#pragma unroll
  for (int j = 0; j <= L2; ++j) {
    if (j > 0) {
#pragma unroll
      for (int i = 0; i <= NM - j; ++i)
#pragma unroll
        for (int m = 0; m <= MM; ++m) T[i][m] = fma(x12, T[i][m], T[i + 1][m]);
    }
    // ket transfer of the rows i <= L1 of this j, in place on a copy
#pragma unroll
    for (int i = 0; i <= L1; ++i) {
      double R[MM + 1];
#pragma unroll
      for (int m = 0; m <= MM; ++m) R[m] = T[i][m];
#pragma unroll
      for (int l = 0; l <= L4; ++l) {
        if (l > 0) {
#pragma unroll
          for (int k = 0; k <= MM - l; ++k) R[k] = fma(x34, R[k], R[k + 1]);
        }
#pragma unroll
        for (int k = 0; k <= L3; ++k) dst[i * s1 + j * s2 + k * s3 + l * s4] = R[k];
      }
    }
  }
}

// Phase 1 in two stages for the eight-warp class (gg|gg) (and three four-warp classes, see CoopTraits::SPLIT1).  With one lane per (root, axis) the 27 lanes that build the 2-D
// integrals work alone while the other 229 wait, and that build -- mostly the ket transfer, 25 values for each of the 25 bra
// index pairs -- is as long as the product phase.  Stage a: lane (root, axis) runs the vertical recurrence and the bra
// transfer and leaves B(i1, i2, m), m = 0..l3+l4, in a scratch area; stage b: the 3 N (l1+1)(l2+1) independent ket transfers
// are dealt over all lanes of the group.  Measured on cfg1 (profiles/r02_cfg1.md): (gg|gg) K = 3 2174 -> 1801 ms (15.8 -> 19.2 %
// of the FP64 peak), K = 1 100.9 -> 93.7 ms; for the four-warp classes the extra shared memory (one block per SM instead of two
// for (gg|gf), (gf|gf): 1530 -> 2345 ms) and the second barrier cost more than the idle lanes, so they keep the one-stage build.
template <int L1, int L2, int MM>
__device__ __forceinline__ void fill_2d_bra(double* __restrict__ scr, double init, double c00, double c00p, double b10, double b01,
                                            double b00, double x12) {
  constexpr int NM = L1 + L2;
  double T[NM + 1][MM + 1];
  T[0][0] = init;
#pragma unroll
  for (int n = 0; n < NM; ++n) T[n + 1][0] = n > 0 ? fma(c00, T[n][0], (n * b10) * T[n - 1][0]) : c00 * T[n][0];
#pragma unroll
  for (int m = 0; m < MM; ++m)
#pragma unroll
    for (int n = 0; n <= NM; ++n) {
      double v = c00p * T[n][m];
      if (m > 0) v = fma(m * b01, T[n][m - 1], v);
      if (n > 0) v = fma(n * b00, T[n - 1][m], v);
      T[n][m + 1] = v;
    }
#pragma unroll
  for (int j = 0; j <= L2; ++j) {
    if (j > 0) {
#pragma unroll
      for (int i = 0; i <= NM - j; ++i)
#pragma unroll
        for (int m = 0; m <= MM; ++m) T[i][m] = fma(x12, T[i][m], T[i + 1][m]);
    }
#pragma unroll
    for (int i = 0; i <= L1; ++i)
#pragma unroll
      for (int m = 0; m <= MM; ++m) scr[(i * (L2 + 1) + j) * (MM + 1) + m] = T[i][m];
  }
}

// one ket transfer: R(m) = B(i1, i2, m) -> I(i1, i2, i3, i4) at dst[i3 * s3 + i4 * s4]
template <int L3, int L4>
__device__ __forceinline__ void ket_transfer(const double* __restrict__ src, double* __restrict__ dst, int s3, int s4, double x34) {
  constexpr int MM = L3 + L4;
  double R[MM + 1];
#pragma unroll
  for (int m = 0; m <= MM; ++m) R[m] = src[m];
#pragma unroll
  for (int l = 0; l <= L4; ++l) {
    if (l > 0) {
#pragma unroll
      for (int k = 0; k <= MM - l; ++k) R[k] = fma(x34, R[k], R[k + 1]);
    }
#pragma unroll
    for (int k = 0; k <= L3; ++k) dst[k * s3 + l * s4] = R[k];
  }
}

__device__ __forceinline__ void cart_powers(int l, int k, int& lx, int& ly, int& lz) {
  int row = 0;
  while ((row + 1) * (row + 2) / 2 <= k) ++row;   // row = l - lx
  lx = l - row;
  ly = row - (k - row * (row + 1) / 2);
  lz = l - lx - ly;
}

__device__ __forceinline__ void group_sync(int tw, int id) {
  if (tw == 1) __syncwarp();
  else asm volatile("bar.sync %0, %1;" ::"r"(id + 1), "r"(32 * tw) : "memory");
}

// NCH > 1: the Cartesian components of shell c are split into NCH chunks and blockIdx.y selects the chunk, so that the
// accumulators per lane, PASSES * (nc(lc) / NCH) * nc(ld), stay in registers for the heaviest classes ((gf|ff) ... (gg|gg));
// the 2-D integrals are then rebuilt once per chunk (cheap next to the products of such classes).
template <int LA, int LB, int LC, int LD, int TW, int NCH = 1>
struct CoopTraits {
  static constexpr int WARPS = TW > COOP_WARPS ? TW : COOP_WARPS;   // TW = 8: the block is one group of eight warps (slab-bound classes)
  static constexpr int T = 32 * TW, GROUPS = WARPS / TW;
  static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC) / NCH, ND = ncart(LD);   // NC: components of c per chunk
  static_assert(ncart(LC) % NCH == 0, "NCH must divide the number of Cartesian components of shell c");
  static constexpr int NAB = NA * NB, NCD = NC * ND;
  static constexpr int PASSES = (NAB + T - 1) / T;
  // three blocks per SM (170 registers) pay off for the classes with 16-20 accumulators per lane (measured on cfg3), not elsewhere
  static constexpr int MINB = (PASSES * NCD >= 16 && PASSES * NCD <= 20) ? 3 : 0;   // 0 = unspecified (the compiler default keeps occupancy higher than an explicit 1)
  static constexpr int N = nroots_of(LA + LB + LC + LD);
  // strides of the slab: SCD = one (i,j) row, G2 = one (axis, root) block; both padded to odd so that lanes that differ in
  // (i,j) (phase 2 loads) or in (axis, root) (phase 1 stores) fall into different shared-memory banks
  static constexpr int SCD = ((LC + 1) * (LD + 1)) | 1, G2 = ((LA + 1) * (LB + 1) * SCD) | 1;
  static constexpr int SLAB2D = 3 * N * G2;
  static constexpr int KROW = (2 * (NC + ND)) | 1;           // per (a,b): Kac[NC] Kad[ND] Kbc[NC] Kbd[ND]; odd stride: no bank conflicts
  static constexpr int SLABK = PASSES * T * KROW;
  // two-stage phase 1 (fill_2d_bra + ket_transfer): the slab-bound class (gg|gg) and the three four-warp classes that measured
  // faster with it on cfg1 K = 3 ((gd|ff) 232 -> 215 ms, (gd|gd) 196 -> 186, (gg|dd) 197 -> 176; (ff|ff) 233 -> 298 and the others slower)
  static constexpr bool SPLIT1 = TW >= 8 || (TW == 4 && LA == 4 && ((LB == 2 && LC == 3 && LD == 3) || (LB == 2 && LC == 4 && LD == 2) || (LB == 4 && LC == 2 && LD == 2)));
  static constexpr int NIJ = (LA + 1) * (LB + 1), MM1 = LC + LD + 1;
  static constexpr int SCR = SPLIT1 ? 3 * N * NIJ * MM1 : 0;    // B(i, j, m) of every (root, axis)
  // paired phase 1 (one-warp classes with at most five roots): the two half-warps build the 2-D integrals of two consecutive
  // primitive quartets of the task at once, each into its own slab; phase 2 then consumes the slabs one after the other.
  // With one lane per (root, axis) phase 1 kept 3 N of 32 lanes busy and took a third of the family's time on cfg3.
  // Not where the second slab would cost a resident block ((ff|dp): 78 -> 132 KB per block, one block per SM instead of two,
  // 8.5 -> 9.9 ms on cfg3): the kernels with 36 or more accumulators per lane hold two blocks per SM by registers, the others three.
  static constexpr int S0 = SLAB2D > SLABK ? SLAB2D : SLABK;                // first slab, later the K partial sums
  static constexpr size_t SMEM_PAIRED = sizeof(double) * (S0 + SLAB2D + NCD) * GROUPS;
  static constexpr bool PAIR = TW == 1 && NCH == 1 && !SPLIT1 && 3 * N <= 16 && SMEM_PAIRED <= (PASSES * NCD >= 36 ? 113 : 75) * 1024;
  static constexpr int SLAB = S0 + (PAIR ? SLAB2D : 0) + SCR + NCD;   // + second slab + bra-transfer scratch + staged D_cd
  static constexpr size_t SMEM = sizeof(double) * SLAB * GROUPS;
  static_assert(SMEM <= 227 * 1024, "cooperative kernel: shared memory");
};

template <int LA, int LB, int LC, int LD, int TW, int NCH = 1>
__global__ void __launch_bounds__(32 * (CoopTraits<LA, LB, LC, LD, TW, NCH>::WARPS), (CoopTraits<LA, LB, LC, LD, TW, NCH>::MINB)) coop_jk_kernel(Work w) {
  using Tr = CoopTraits<LA, LB, LC, LD, TW, NCH>;
  constexpr int T = Tr::T, GROUPS = Tr::GROUPS;
  constexpr int NA = Tr::NA, NB = Tr::NB, NC = Tr::NC, ND = Tr::ND, NAB = Tr::NAB, NCD = Tr::NCD, PASSES = Tr::PASSES;
  constexpr int N = Tr::N, SCD = Tr::SCD, G2 = Tr::G2;
  extern __shared__ double smem[];
  const int lane = threadIdx.x, wy = threadIdx.y;   // lane: thread within the group of T; wy: group within the block
  double* S = smem + (size_t)wy * Tr::SLAB;      // 2-D integrals, later the K partial sums
  double* sDcd = S + (Tr::SLAB - NCD);             // D_cd of the task's ket pair
  [[maybe_unused]] double* scr = S + (Tr::SLAB - NCD - Tr::SCR);   // two-stage phase 1: B(i, j, m) per (root, axis)

  const PairSet& bp = w.bra; const PairSet& kp = w.ket;
  const int blk = blockIdx.x * w.nshard + w.shard;
  const bool list = w.list != nullptr;
  int i_begin, i_end, j;
  if (list) {
    const long t = (long)blk * GROUPS + wy;
    if (t >= w.nlist) return;
    i_begin = w.list[t].x; i_end = i_begin + 1; j = w.list[t].y;
  } else {
    if (blk >= w.row_off[w.nrows]) return;
    const int r = find_row_warp(w.row_off, w.nrows, blk, threadIdx.x & 31);
    j = (blk - w.row_off[r]) * GROUPS + wy;
    i_begin = r * COOP_CH; i_end = min(i_begin + COOP_CH, bp.npair);
    if (j >= kp.npair) return;
  }
  const int n = w.nao;
  const double* __restrict__ D = w.D;

  // ---- per-task ket data ------------------------------------------------------------------------------------------
  double C[3], CD[3];
#pragma unroll
  for (int x = 0; x < 3; ++x) { C[x] = kp.geom[x * kp.stride + j]; CD[x] = kp.geom[(3 + x) * kp.stride + j]; }
  const double wket = kp.geom[6 * kp.stride + j];
  const int c_lo = NCH > 1 ? (int)blockIdx.y * NC : 0;   // first component of this block's chunk of shell c
  const int c0 = kp.ao[j].x + c_lo, d0 = kp.ao[j].y;     // everything below addresses D, J, K through c0: chunk-local c
  for (int cd = lane; cd < NCD; cd += T) sDcd[cd] = D[(long)(c0 + cd / ND) * n + d0 + cd % ND];
  group_sync(TW, wy);
  int ocx[NCH > 1 ? NC : 1], ocy[NCH > 1 ? NC : 1], ocz[NCH > 1 ? NC : 1];   // slab offsets of the chunk's components (NCH > 1)
  if (NCH > 1) {
#pragma unroll
    for (int cl = 0; cl < NC; ++cl) {
      int px, py, pz;
      cart_powers(LC, c_lo + cl, px, py, pz);
      ocx[cl] = px * (LD + 1); ocy[cl] = py * (LD + 1); ocz[cl] = pz * (LD + 1);
    }
  }

  // ---- per-lane roles ---------------------------------------------------------------------------------------------
  // phase 1: lane -> (root, axis)
  const int my_root = lane / 3, my_axis = lane - 3 * my_root;
  const bool fill_lane = lane < 3 * N;
  // phase 2: lane -> bra component pairs ab = lane + T*pass
  int offx[PASSES], offy[PASSES], offz[PASSES], ia[PASSES], ib[PASSES];
#pragma unroll
  for (int ps = 0; ps < PASSES; ++ps) {
    int ab = lane + T * ps;
    if (ab >= NAB) ab = NAB - 1;   // idle lanes of the last pass compute a duplicate that is never written out
    ia[ps] = ab / NB; ib[ps] = ab - ia[ps] * NB;
    int ax, ay, az, bx, by, bz;
    cart_powers(LA, ia[ps], ax, ay, az); cart_powers(LB, ib[ps], bx, by, bz);
    offx[ps] = (ax * (LB + 1) + bx) * SCD;
    offy[ps] = (ay * (LB + 1) + by) * SCD + N * G2;
    offz[ps] = (az * (LB + 1) + bz) * SCD + 2 * N * G2;
  }
  double pjcd[NCD];
#pragma unroll
  for (int cd = 0; cd < NCD; ++cd) pjcd[cd] = 0.0;
  double g[PASSES][NCD];
#pragma unroll
  for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
    for (int cd = 0; cd < NCD; ++cd) g[ps][cd] = 0.0;

  // ---- phase 2: g[ab][cd] += sum over the roots of X Y Z from the slab S2 --------------------------------------------
  auto phase2 = [&](const double* __restrict__ S2) {
#pragma unroll 1
    for (int r = 0; r < N; ++r) {
#pragma unroll
      for (int ps = 0; ps < PASSES; ++ps) {
        const double* X = S2 + offx[ps] + r * G2;
        const double* Y = S2 + offy[ps] + r * G2;
        const double* Z = S2 + offz[ps] + r * G2;
        if constexpr (NCH > 1) {
#pragma unroll
          for (int cl = 0; cl < NC; ++cl) {
            int d = 0;
#pragma unroll
            for (int dx = LD; dx >= 0; --dx)
#pragma unroll
            for (int dy = LD - dx; dy >= 0; --dy) {
              const int dz = LD - dx - dy;
              g[ps][cl * ND + d] = fma(X[ocx[cl] + dx] * Y[ocy[cl] + dy], Z[ocz[cl] + dz], g[ps][cl * ND + d]);
              ++d;
            }
          }
        } else {
        int cd = 0;
#pragma unroll
        for (int cx = LC; cx >= 0; --cx)
#pragma unroll
        for (int cy = LC - cx; cy >= 0; --cy)
#pragma unroll
        for (int dx = LD; dx >= 0; --dx)
#pragma unroll
        for (int dy = LD - dx; dy >= 0; --dy) {
          const int cz = LC - cx - cy, dz = LD - dx - dy;
          g[ps][cd] = fma(X[cx * (LD + 1) + dx] * Y[cy * (LD + 1) + dy], Z[cz * (LD + 1) + dz], g[ps][cd]);
          ++cd;
        }
        }
      }
    }
  };

  // ---- phase 3: digestion of the finished quartet (bra pair i, ket pair j), then g = 0 ---------------------------------
  auto phase3 = [&](int i, double f) {
    const int a0 = bp.ao[i].x, b0 = bp.ao[i].y;
#pragma unroll
    for (int ps = 0; ps < PASSES; ++ps) {
      const bool own = lane + T * ps < NAB;
      const long ra = (long)(a0 + ia[ps]) * n, rb = (long)(b0 + ib[ps]) * n;
      // D is symmetric (eri.h): the blocks are read through their transposes, D_ca, D_cb, D_da, D_db, so that the lanes of one
      // load instruction -- fixed c or d, bra components a or b across the lanes -- touch one row of D instead of NA or NB rows
      const int ca = a0 + ia[ps], cb = b0 + ib[ps];
      const double Dab = own ? f * D[rb + ca] : 0.0;
      const double fo = own ? f : 0.0;
      double Dac[NC], Dbc[NC], Dad[ND], Dbd[ND];
#pragma unroll
      for (int c = 0; c < NC; ++c) { const long rc = (long)(c0 + c) * n; Dac[c] = D[rc + ca]; Dbc[c] = D[rc + cb]; }
#pragma unroll
      for (int d = 0; d < ND; ++d) { const long rd = (long)(d0 + d) * n; Dad[d] = D[rd + ca]; Dbd[d] = D[rd + cb]; }
      double jab = 0.0, kac[NC], kbc[NC], kad[ND], kbd[ND];
#pragma unroll
      for (int c = 0; c < NC; ++c) kac[c] = kbc[c] = 0.0;
#pragma unroll
      for (int d = 0; d < ND; ++d) kad[d] = kbd[d] = 0.0;
#pragma unroll
      for (int c = 0; c < NC; ++c)
#pragma unroll
        for (int d = 0; d < ND; ++d) {
          const double v = g[ps][c * ND + d];
          jab = fma(v, sDcd[c * ND + d], jab);
          pjcd[c * ND + d] = fma(v, Dab, pjcd[c * ND + d]);
          kac[c] = fma(v, Dbd[d], kac[c]);
          kad[d] = fma(v, Dbc[c], kad[d]);
          kbc[c] = fma(v, Dad[d], kbc[c]);
          kbd[d] = fma(v, Dac[c], kbd[d]);
        }
      if (own) atomic_add(w.J + ra + b0 + ib[ps], fo * jab);
      double* row = S + (size_t)(lane + T * ps) * Tr::KROW;
#pragma unroll
      for (int c = 0; c < NC; ++c) { row[c] = fo * kac[c]; row[NC + ND + c] = fo * kbc[c]; }
#pragma unroll
      for (int d = 0; d < ND; ++d) { row[NC + d] = fo * kad[d]; row[2 * NC + ND + d] = fo * kbd[d]; }
    }
    group_sync(TW, wy);
    // K_a. = sum over b of the rows (a,b); K_b. = sum over a.  Items: [a][NC+ND] then [b][NC+ND].
    for (int it = lane; it < (NA + NB) * (NC + ND); it += T) {
      const bool isa = it < NA * (NC + ND);
      const int rem = isa ? it : it - NA * (NC + ND);
      const int s = rem / (NC + ND), e = rem - s * (NC + ND);    // s = a or b; e < NC: column c, else column d
      double sum = 0.0;
      if (isa) { for (int b = 0; b < NB; ++b) sum += S[(size_t)(s * NB + b) * Tr::KROW + e]; }
      else     { for (int a = 0; a < NA; ++a) sum += S[(size_t)(a * NB + s) * Tr::KROW + (NC + ND) + e]; }
      const long rowK = (long)((isa ? a0 : b0) + s) * n;
      const int col = e < NC ? c0 + e : d0 + (e - NC);
      atomic_add(w.K + rowK + col, sum);
    }
    group_sync(TW, wy);
#pragma unroll
    for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
      for (int cd = 0; cd < NCD; ++cd) g[ps][cd] = 0.0;
  };

  if constexpr (!Tr::PAIR) {
  for (int i = i_begin; i < i_end; ++i) {
    double f;
    if (list) f = 1.0;
    else {
      if (j >= w.ket_count[i]) continue;     // warp-uniform
      f = bp.geom[6 * bp.stride + i] * wket;
      if (w.same && i == j) f *= 0.5;
    }
    double A[3], AB[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) { A[x] = bp.geom[x * bp.stride + i]; AB[x] = bp.geom[(3 + x) * bp.stride + i]; }

    for (int kb = 0; kb < bp.npp; ++kb) {
      const double p = bp.prim[(kb * 5 + 0) * bp.stride + i];
      const double P[3] = {bp.prim[(kb * 5 + 1) * bp.stride + i], bp.prim[(kb * 5 + 2) * bp.stride + i], bp.prim[(kb * 5 + 3) * bp.stride + i]};
      const double Kab = bp.prim[(kb * 5 + 4) * bp.stride + i];
      // build on B when P is nearer to B (only if there is something to transfer)
      bool swb = false;
      if (LB > 0) {
        double da = 0.0, db = 0.0;
#pragma unroll
        for (int x = 0; x < 3; ++x) { const double pa = P[x] - A[x], pb = pa + AB[x]; da += pa * pa; db += pb * pb; }
        swb = db < da;
      }
      for (int kk = 0; kk < kp.npp; ++kk) {
        const double q = kp.prim[(kk * 5 + 0) * kp.stride + j];
        const double Q[3] = {kp.prim[(kk * 5 + 1) * kp.stride + j], kp.prim[(kk * 5 + 2) * kp.stride + j], kp.prim[(kk * 5 + 3) * kp.stride + j]};
        const double Kcd = kp.prim[(kk * 5 + 4) * kp.stride + j];
        bool swk = false;
        if (LD > 0) {
          double dc = 0.0, dd = 0.0;
#pragma unroll
          for (int x = 0; x < 3; ++x) { const double qc = Q[x] - C[x], qd = qc + CD[x]; dc += qc * qc; dd += qd * qd; }
          swk = dd < dc;
        }
        const double rpq = 1.0 / (p + q), rho = p * q * rpq;
        const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
        const double x = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
        // ---- phase 1 ----
        if constexpr (Tr::SPLIT1) {
          constexpr int NIJ = Tr::NIJ, MM1 = Tr::MM1;
          constexpr int SI = (LB + 1) * SCD, SJ = SCD, SK = LD + 1, SL = 1;
          const double cdx3[3] = {CD[0], CD[1], CD[2]};
          if (fill_lane) {   // stage a: vertical recurrence + bra transfer
            double u, wt;
            rys_root_one<N>(x, w.rys, my_root, u, wt);
            const double t2 = u * rpq;
            const double b00 = 0.5 * t2, b10 = (1.0 - q * t2) * 0.5 / p, b01 = (1.0 - p * t2) * 0.5 / q;
            const int ax = my_axis;
            const double pa = (ax == 0 ? P[0] - A[0] : ax == 1 ? P[1] - A[1] : P[2] - A[2]);
            const double qc = (ax == 0 ? Q[0] - C[0] : ax == 1 ? Q[1] - C[1] : Q[2] - C[2]);
            const double pqx = (ax == 0 ? PQ[0] : ax == 1 ? PQ[1] : PQ[2]);
            const double abx = (ax == 0 ? AB[0] : ax == 1 ? AB[1] : AB[2]);
            const double cdx = cdx3[ax];
            const double c00 = pa + (swb ? abx : 0.0) - q * t2 * pqx;
            const double c00p = qc + (swk ? cdx : 0.0) + p * t2 * pqx;
            const double init = ax == 2 ? Kab * Kcd * sqrt(rpq) * wt : 1.0;
            double* dsts = scr + (ax * N + my_root) * (NIJ * MM1);   // B(i1, i2, m): i1 on the build centre
            if (!swb) fill_2d_bra<LA, LB, LC + LD>(dsts, init, c00, c00p, b10, b01, b00, abx);
            else if constexpr (LB > 0) fill_2d_bra<LB, LA, LC + LD>(dsts, init, c00, c00p, b10, b01, b00, -abx);
          }
          group_sync(TW, wy);
          // stage b: ket transfers, one per (root, axis, i1, i2), over all lanes of the group
          for (int tk = lane; tk < 3 * N * NIJ; tk += T) {
            const int ra = tk / NIJ, ij = tk - ra * NIJ, ax = ra / N;   // ra = axis * N + root
            const double* src = scr + (size_t)tk * MM1;
            // (i1, i2) -> (i, j) of the slab: built on A: i1 = i, i2 = j; built on B: i1 = j, i2 = i
            int i1, i2, off;
            if (!swb) { i1 = ij / (LB + 1); i2 = ij - i1 * (LB + 1); off = i1 * SI + i2 * SJ; }
            else      { i1 = ij / (LA + 1); i2 = ij - i1 * (LA + 1); off = i2 * SI + i1 * SJ; }
            double* dst = S + ra * G2 + off;
            if (!swk) ket_transfer<LC, LD>(src, dst, SK, SL, cdx3[ax]);
            else if constexpr (LD > 0) ket_transfer<LD, LC>(src, dst, SL, SK, -cdx3[ax]);
          }
        } else
        if (fill_lane) {
          double u, wt;
          rys_root_one<N>(x, w.rys, my_root, u, wt);
          const double t2 = u * rpq;
          const double b00 = 0.5 * t2, b10 = (1.0 - q * t2) * 0.5 / p, b01 = (1.0 - p * t2) * 0.5 / q;
          const int ax = my_axis;
          const double pa = (ax == 0 ? P[0] - A[0] : ax == 1 ? P[1] - A[1] : P[2] - A[2]);
          const double qc = (ax == 0 ? Q[0] - C[0] : ax == 1 ? Q[1] - C[1] : Q[2] - C[2]);
          const double pqx = (ax == 0 ? PQ[0] : ax == 1 ? PQ[1] : PQ[2]);
          const double abx = (ax == 0 ? AB[0] : ax == 1 ? AB[1] : AB[2]);
          const double cdx = (ax == 0 ? CD[0] : ax == 1 ? CD[1] : CD[2]);
          const double c00 = pa + (swb ? abx : 0.0) - q * t2 * pqx;
          const double c00p = qc + (swk ? cdx : 0.0) + p * t2 * pqx;
          const double init = ax == 2 ? Kab * Kcd * sqrt(rpq) * wt : 1.0;
          double* dst = S + (ax * N + my_root) * G2;
          constexpr int SI = (LB + 1) * SCD, SJ = SCD, SK = LD + 1, SL = 1;
          if (!swb) {
            if (!swk) fill_2d_smem<LA, LB, LC, LD>(dst, SI, SJ, SK, SL, init, c00, c00p, b10, b01, b00, abx, cdx);
            else if constexpr (LD > 0) fill_2d_smem<LA, LB, LD, LC>(dst, SI, SJ, SL, SK, init, c00, c00p, b10, b01, b00, abx, -cdx);
          } else if constexpr (LB > 0) {
            if (!swk) fill_2d_smem<LB, LA, LC, LD>(dst, SJ, SI, SK, SL, init, c00, c00p, b10, b01, b00, -abx, cdx);
            else if constexpr (LD > 0) fill_2d_smem<LB, LA, LD, LC>(dst, SJ, SI, SL, SK, init, c00, c00p, b10, b01, b00, -abx, -cdx);
          }
        }
        group_sync(TW, wy);
        phase2(S);
        group_sync(TW, wy);
      }
    }

    phase3(i, f);
  }

  } else {
  // ---- paired phase 1: the primitive quartets of the task (bra pair, bra primitive pair, ket primitive pair) are walked two
  // at a time; half-warp h builds item h into slab h with its lanes (root, axis), phase 2 consumes slab 0, then slab 1, and a
  // quartet is digested as soon as its last primitive quartet has been added.
  const int h = lane >> 4, hl = lane & 15;
  const int p_root = hl / 3, p_axis = hl - 3 * p_root;
  const bool p_fill = hl < 3 * N;
  const unsigned team = ((1u << (3 * N)) - 1u) << (16 * h);
  double* Sh = S + h * Tr::S0;
  const int nkb = bp.npp, nkk = kp.npp;
  auto has_work = [&](int i) { return list || j < w.ket_count[i]; };   // warp-uniform
  auto weight = [&](int i) {
    if (list) return 1.0;
    double f = bp.geom[6 * bp.stride + i] * wket;
    if (w.same && i == j) f *= 0.5;
    return f;
  };
  int i0 = i_begin;
  while (i0 < i_end && !has_work(i0)) ++i0;
  int kb0 = 0, kk0 = 0;
  while (i0 < i_end) {
    // second item of the pair: the next primitive quartet of the task
    int i1 = i0, kb1 = kb0, kk1 = kk0 + 1;
    if (kk1 == nkk) { kk1 = 0; if (++kb1 == nkb) { kb1 = 0; ++i1; while (i1 < i_end && !has_work(i1)) ++i1; } }
    const int mi = h ? i1 : i0, mkb = h ? kb1 : kb0, mkk = h ? kk1 : kk0;
    if (p_fill && mi < i_end) {
      double A[3], AB[3];
#pragma unroll
      for (int x = 0; x < 3; ++x) { A[x] = bp.geom[x * bp.stride + mi]; AB[x] = bp.geom[(3 + x) * bp.stride + mi]; }
      const double p = bp.prim[(mkb * 5 + 0) * bp.stride + mi];
      const double P[3] = {bp.prim[(mkb * 5 + 1) * bp.stride + mi], bp.prim[(mkb * 5 + 2) * bp.stride + mi], bp.prim[(mkb * 5 + 3) * bp.stride + mi]};
      const double Kab = bp.prim[(mkb * 5 + 4) * bp.stride + mi];
      bool swb = false;   // build on B when P is nearer to B (only if there is something to transfer)
      if (LB > 0) {
        double da = 0.0, db = 0.0;
#pragma unroll
        for (int x = 0; x < 3; ++x) { const double pa = P[x] - A[x], pb = pa + AB[x]; da += pa * pa; db += pb * pb; }
        swb = db < da;
      }
      const double q = kp.prim[(mkk * 5 + 0) * kp.stride + j];
      const double Q[3] = {kp.prim[(mkk * 5 + 1) * kp.stride + j], kp.prim[(mkk * 5 + 2) * kp.stride + j], kp.prim[(mkk * 5 + 3) * kp.stride + j]};
      const double Kcd = kp.prim[(mkk * 5 + 4) * kp.stride + j];
      bool swk = false;
      if (LD > 0) {
        double dc = 0.0, dd = 0.0;
#pragma unroll
        for (int x = 0; x < 3; ++x) { const double qc = Q[x] - C[x], qd = qc + CD[x]; dc += qc * qc; dd += qd * qd; }
        swk = dd < dc;
      }
      const double rpq = 1.0 / (p + q), rho = p * q * rpq;
      const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
      const double x = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
      double u, wt;
      rys_root_team<N>(x, w.rys, p_root, p_axis, 16 * h, team, u, wt);
      const double t2 = u * rpq;
      const double b00 = 0.5 * t2, b10 = (1.0 - q * t2) * 0.5 / p, b01 = (1.0 - p * t2) * 0.5 / q;
      const int ax = p_axis;
      const double pa = (ax == 0 ? P[0] - A[0] : ax == 1 ? P[1] - A[1] : P[2] - A[2]);
      const double qc = (ax == 0 ? Q[0] - C[0] : ax == 1 ? Q[1] - C[1] : Q[2] - C[2]);
      const double pqx = (ax == 0 ? PQ[0] : ax == 1 ? PQ[1] : PQ[2]);
      const double abx = (ax == 0 ? AB[0] : ax == 1 ? AB[1] : AB[2]);
      const double cdx = (ax == 0 ? CD[0] : ax == 1 ? CD[1] : CD[2]);
      const double c00 = pa + (swb ? abx : 0.0) - q * t2 * pqx;
      const double c00p = qc + (swk ? cdx : 0.0) + p * t2 * pqx;
      const double init = ax == 2 ? Kab * Kcd * sqrt(rpq) * wt : 1.0;
      double* dst = Sh + (ax * N + p_root) * G2;
      constexpr int SI = (LB + 1) * SCD, SJ = SCD, SK = LD + 1, SL = 1;
      if (!swb) {
        if (!swk) fill_2d_smem<LA, LB, LC, LD>(dst, SI, SJ, SK, SL, init, c00, c00p, b10, b01, b00, abx, cdx);
        else if constexpr (LD > 0) fill_2d_smem<LA, LB, LD, LC>(dst, SI, SJ, SL, SK, init, c00, c00p, b10, b01, b00, abx, -cdx);
      } else if constexpr (LB > 0) {
        if (!swk) fill_2d_smem<LB, LA, LC, LD>(dst, SJ, SI, SK, SL, init, c00, c00p, b10, b01, b00, -abx, cdx);
        else if constexpr (LD > 0) fill_2d_smem<LB, LA, LD, LC>(dst, SJ, SI, SL, SK, init, c00, c00p, b10, b01, b00, -abx, -cdx);
      }
    }
    __syncwarp();
#pragma unroll 1
    for (int t = 0; t < 2; ++t) {   // (not unrolled: one copy of the phase 2 and phase 3 code)
      const int ti = t ? i1 : i0;
      if (ti >= i_end) break;
      phase2(S + t * Tr::S0);
      // slab 0 is dead by now: phase 3 keeps the K partial sums there, slab 1 stays untouched
      if ((t ? kb1 : kb0) == nkb - 1 && (t ? kk1 : kk0) == nkk - 1) phase3(ti, weight(ti));
    }
    __syncwarp();
    // first item of the next pair
    i0 = i1; kb0 = kb1; kk0 = kk1 + 1;
    if (i0 < i_end && kk0 == nkk) { kk0 = 0; if (++kb0 == nkb) { kb0 = 0; ++i0; while (i0 < i_end && !has_work(i0)) ++i0; } }
  }
  }
  // ---- J_cd of the task: sum the per-lane partial sums over the lanes ------------------------------------------------
#pragma unroll
  for (int cd = 0; cd < NCD; ++cd) {
    double s = pjcd[cd];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((lane & 31) == (cd & 31) && s != 0.0) atomic_add(w.J + (long)(c0 + cd / ND) * n + d0 + cd % ND, s);
  }
}

template <int LA, int LB, int LC, int LD, int TW, int NCH = 1>
cudaError_t launch_coop_jk(const Work& w, int nblocks_dense, cudaStream_t s) {
  using Tr = CoopTraits<LA, LB, LC, LD, TW, NCH>;
  const int total = w.list ? (w.nlist + Tr::GROUPS - 1) / Tr::GROUPS : nblocks_dense;
  const int grid = (total + w.nshard - 1) / w.nshard;
  if (grid <= 0) return cudaSuccess;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(coop_jk_kernel<LA, LB, LC, LD, TW, NCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tr::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  coop_jk_kernel<LA, LB, LC, LD, TW, NCH><<<dim3(grid, NCH), dim3(Tr::T, Tr::GROUPS), Tr::SMEM, s>>>(w);
  return cudaGetLastError();
}

}  // namespace eri
