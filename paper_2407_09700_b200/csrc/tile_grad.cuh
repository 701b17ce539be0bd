// tile_grad.cuh -- tile family, J/K gradient kernel (Algorithm 4; Eq. 11-15).
// Same tiling as tile_kernel.cuh (block = bra chunk x ket chunk of the grouped pair sets, a warp walks down the bra rows,
// lane = ket slot), one thread per quartet.  Per root the 2-D integrals are built in registers with every index that is
// differentiated raised by one (centres A, B, C; centre D follows from translational invariance), and each
// Cartesian element contributes  dI/dR . (PJ, PK)  straight into 18 per-thread scalars (reading R10/R11:
// PJ = 4 f D_ab D_cd, PK = 2 f (D_ab' ...) = 2 f (D_ac D_bd + D_ad D_bc)) -- there is no per-element accumulator, so the
// footprint does not grow with Pi nc(l).  The six density blocks of a quartet are staged in shared memory: the three
// that do not depend on the ket's second shell (D_ab once per warp; D_ac, D_bc once per ket half), the three that do
// (D_cd, D_ad, D_bd) in a column per lane.  The 18 scalars are summed over the lanes through the warp's
// shared-memory transpose and leave as at most 36 FP64 atomics per ROW (one sum per ket half) (the paper: 12 atomics per quartet);
// the centre-D part is kept per lane over the rows and leaves once per block.
#pragma once
#include "tile_kernel.cuh"

namespace eri {

template <int LA, int LB, int LC, int LD, int BI, int MODE = 0>
struct TileGradTraits {
  static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
  static constexpr int N = nroots_of(LA + LB + LC + LD + 1);
  static constexpr int G2 = (LA + 2) * (LB + 2) * (LC + 2) * (LD + 1);          // raised on A, B, C
  static constexpr int NUNI = NA * NB + 2 * (NA * NC + NB * NC);                 // D_ab per warp; D_ac, D_bc per ket half
  static constexpr int NLANE = NC * ND + NA * ND + NB * ND;                       // D_cd, D_ad, D_bd: per lane
  static constexpr int STAGE = 32 * 33;
  static constexpr int NE = NA * NB * NC * ND;
  static constexpr int PERWARP = STAGE + NUNI + 32 * NLANE;
  static constexpr int RT = rys2_size(N);                    // the class's Rys table, first in the block's shared memory
  static constexpr size_t SMEM = sizeof(double) * (RT + BI * PERWARP);
};

// One differentiated axis AX of one root (MODE 1): the 2-D integrals of axis AX are built raised on A, B, C, those of the
// other two axes plain, so that only (LA+2)(LB+2)(LC+2)(LD+1) + 2 (LA+1)(LB+1)(LC+1)(LD+1) words are live at a time.
// c00[3], c00p[3]: the recurrence constants per axis; init[3]: 1, 1, prefactor x weight.
template <int LA, int LB, int LC, int LD, int AX>
__device__ __forceinline__ void tile_grad_axis(double* __restrict__ acc, const double* c00, const double* c00p, const double* init,
                                               double b10, double b01, double b00, const double* AB, const double* CD,
                                               double ea2, double eb2, double ec2,
                                               const double* Dab_s, const double* Dac_s, const double* Dbc_s,
                                               const double* Dcd_s, const double* Dad_s, const double* Dbd_s) {
  constexpr int NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
  constexpr int G2R = (LA + 2) * (LB + 2) * (LC + 2) * (LD + 1), G2B = (LA + 1) * (LB + 1) * (LC + 1) * (LD + 1);
  constexpr int RC = LD + 1, RB = (LC + 2) * RC, RA = (LB + 2) * RB;     // raised strides
  constexpr int PC = LD + 1, PB = (LC + 1) * PC, PA = (LB + 1) * PB;     // plain strides
  constexpr int O1 = (AX + 1) % 3, O2 = (AX + 2) % 3;
  double gr[G2R], g1[G2B], g2[G2B];
  fill_2d_tile<LA + 1, LB + 1, LC + 1, LD>(gr, init[AX], c00[AX], c00p[AX], b10, b01, b00, AB[AX], CD[AX]);
  fill_2d_tile<LA, LB, LC, LD>(g1, init[O1], c00[O1], c00p[O1], b10, b01, b00, AB[O1], CD[O1]);
  fill_2d_tile<LA, LB, LC, LD>(g2, init[O2], c00[O2], c00p[O2], b10, b01, b00, AB[O2], CD[O2]);
  int a = 0;
#pragma unroll
  for (int ax = LA; ax >= 0; --ax)
#pragma unroll
  for (int ay = LA - ax; ay >= 0; --ay) {
    const int pa[3] = {ax, ay, LA - ax - ay};
    int b = 0;
#pragma unroll
    for (int bx = LB; bx >= 0; --bx)
#pragma unroll
    for (int by = LB - bx; by >= 0; --by) {
      const int pb[3] = {bx, by, LB - bx - by};
      const double dab = Dab_s[a * NB + b];
      int c = 0;
#pragma unroll
      for (int cx = LC; cx >= 0; --cx)
#pragma unroll
      for (int cy = LC - cx; cy >= 0; --cy) {
        const int pc[3] = {cx, cy, LC - cx - cy};
        const double dac = Dac_s[a * NC + c], dbc = Dbc_s[b * NC + c];
        int d = 0;
#pragma unroll
        for (int dx = LD; dx >= 0; --dx)
#pragma unroll
        for (int dy = LD - dx; dy >= 0; --dy) {
          const int pd[3] = {dx, dy, LD - dx - dy};
          const double pj = dab * Dcd_s[32 * (c * ND + d)];
          const double pk = fma(dac, Dbd_s[32 * (b * ND + d)], Dad_s[32 * (a * ND + d)] * dbc);
          const int er = pa[AX] * RA + pb[AX] * RB + pc[AX] * RC + pd[AX];
          const double oth = g1[pa[O1] * PA + pb[O1] * PB + pc[O1] * PC + pd[O1]] * g2[pa[O2] * PA + pb[O2] * PB + pc[O2] * PC + pd[O2]];
          const double dA = pa[AX] > 0 ? fma(ea2, gr[er + RA], -pa[AX] * gr[er - RA]) : ea2 * gr[er + RA];
          const double dB = pb[AX] > 0 ? fma(eb2, gr[er + RB], -pb[AX] * gr[er - RB]) : eb2 * gr[er + RB];
          const double dC = pc[AX] > 0 ? fma(ec2, gr[er + RC], -pc[AX] * gr[er - RC]) : ec2 * gr[er + RC];
          const double tj = pj * oth, tk = pk * oth;
          acc[AX] = fma(dA, tj, acc[AX]); acc[3 + AX] = fma(dB, tj, acc[3 + AX]); acc[6 + AX] = fma(dC, tj, acc[6 + AX]);
          acc[9 + AX] = fma(dA, tk, acc[9 + AX]); acc[12 + AX] = fma(dB, tk, acc[12 + AX]); acc[15 + AX] = fma(dC, tk, acc[15 + AX]);
          ++d;
        }
        ++c;
      }
      ++b;
    }
    ++a;
  }
}

// one differentiated axis of one root with the density products pj[e], pk[e] of the quartet read from a shared-memory column
// (pjk[STRIDE e], pjk[STRIDE (NE + e)]; STRIDE 32: a column per lane, 1: one array per warp); accumulates [J: A, B, C | K: A, B, C] of axis AX
template <int LA, int LB, int LC, int LD, int AX, int STRIDE = 32>
__device__ __forceinline__ void tile_grad_team_axis(double* __restrict__ acc, const double* c00, const double* c00p, const double* init,
                                                    double b10, double b01, double b00, const double* AB, const double* CD,
                                                    double ea2, double eb2, double ec2, const double* __restrict__ pjk) {
  constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD), NE = NA * NB * NC * ND;
  constexpr int G2R = (LA + 2) * (LB + 2) * (LC + 2) * (LD + 1), G2B = (LA + 1) * (LB + 1) * (LC + 1) * (LD + 1);
  constexpr int RC = LD + 1, RB = (LC + 2) * RC, RA = (LB + 2) * RB;     // raised strides
  constexpr int PC = LD + 1, PB = (LC + 1) * PC, PA = (LB + 1) * PB;     // plain strides
  constexpr int O1 = (AX + 1) % 3, O2 = (AX + 2) % 3;
  double gr[G2R], g1[G2B], g2[G2B];
  fill_2d_tile<LA + 1, LB + 1, LC + 1, LD>(gr, init[AX], c00[AX], c00p[AX], b10, b01, b00, AB[AX], CD[AX]);
  fill_2d_tile<LA, LB, LC, LD>(g1, init[O1], c00[O1], c00p[O1], b10, b01, b00, AB[O1], CD[O1]);
  fill_2d_tile<LA, LB, LC, LD>(g2, init[O2], c00[O2], c00p[O2], b10, b01, b00, AB[O2], CD[O2]);
  int e = 0;
#pragma unroll
  for (int ax = LA; ax >= 0; --ax)
#pragma unroll
  for (int ay = LA - ax; ay >= 0; --ay) {
    const int pa[3] = {ax, ay, LA - ax - ay};
#pragma unroll
    for (int bx = LB; bx >= 0; --bx)
#pragma unroll
    for (int by = LB - bx; by >= 0; --by) {
      const int pb[3] = {bx, by, LB - bx - by};
#pragma unroll
      for (int cx = LC; cx >= 0; --cx)
#pragma unroll
      for (int cy = LC - cx; cy >= 0; --cy) {
        const int pc[3] = {cx, cy, LC - cx - cy};
#pragma unroll
        for (int dx = LD; dx >= 0; --dx)
#pragma unroll
        for (int dy = LD - dx; dy >= 0; --dy) {
          const int pd[3] = {dx, dy, LD - dx - dy};
          const int er = pa[AX] * RA + pb[AX] * RB + pc[AX] * RC + pd[AX];
          const double oth = g1[pa[O1] * PA + pb[O1] * PB + pc[O1] * PC + pd[O1]] * g2[pa[O2] * PA + pb[O2] * PB + pc[O2] * PC + pd[O2]];
          const double dA = pa[AX] > 0 ? fma(ea2, gr[er + RA], -pa[AX] * gr[er - RA]) : ea2 * gr[er + RA];
          const double dB = pb[AX] > 0 ? fma(eb2, gr[er + RB], -pb[AX] * gr[er - RB]) : eb2 * gr[er + RB];
          const double dC = pc[AX] > 0 ? fma(ec2, gr[er + RC], -pc[AX] * gr[er - RC]) : ec2 * gr[er + RC];
          const double tj = pjk[STRIDE * e] * oth, tk = pjk[STRIDE * (NE + e)] * oth;
          acc[0] = fma(dA, tj, acc[0]); acc[1] = fma(dB, tj, acc[1]); acc[2] = fma(dC, tj, acc[2]);
          acc[3] = fma(dA, tk, acc[3]); acc[4] = fma(dB, tk, acc[4]); acc[5] = fma(dC, tk, acc[5]);
          ++e;
        }
      }
    }
  }
}

template <int LA, int LB, int LC, int LD, int BI, int MODE>
__global__ void __launch_bounds__(32 * BI) tile_grad_kernel(Work w) {
  using Tr = TileGradTraits<LA, LB, LC, LD, BI, MODE>;
  constexpr int NA = Tr::NA, NB = Tr::NB, NC = Tr::NC, ND = Tr::ND, N = Tr::N, G2 = Tr::G2;
  constexpr int SD = 1, SC = LD + 1, SB = (LC + 2) * SC, SA = (LB + 2) * SB;   // strides of the raised 2-D arrays
  extern __shared__ __align__(16) double smem[];

  const PairSet& bp = w.bra; const PairSet& kp = w.ket;
  const int blk = blockIdx.x * w.nshard + w.shard;
  if (blk >= w.row_off[w.nrows]) return;
  const int r = find_row_warp(w.row_off, w.nrows, blk, threadIdx.x);
  const int x = threadIdx.x, gq = threadIdx.y;
  const int i_first = w.row_slot[r], j_first = (blk - w.row_off[r]) * 32;
  const double* rtab = smem;                       // Rys table of the class (eri_dev.cuh "Shared-memory copy")
  rys_stage_table<N>(smem, w.rys, gq * 32 + x, 32 * BI);
  __syncthreads();
  double* stage = smem + Tr::RT + gq * Tr::PERWARP;
  double* uni = stage + Tr::STAGE;                 // [D_ab | D_ac | D_bc], the same for all lanes
  double* mine = uni + Tr::NUNI + x;               // column of this lane, stride 32: [D_cd | D_ad | D_bd]
  const int half = x >> 4;                         // ket half of this lane: its own shell c
  double* Dab_s = uni; double* Dac_s = uni + NA * NB + half * (NA * NC + NB * NC); double* Dbc_s = Dac_s + NA * NC;
  double* Dcd_s = mine; double* Dad_s = mine + 32 * NC * ND; double* Dbd_s = Dad_s + 32 * NA * ND;

  const int j = j_first + x;
  const double qj = kp.q[j];
  double qk_max = qj;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) qk_max = fmax(qk_max, __shfl_xor_sync(0xffffffffu, qk_max, o));
  const int2 cd0 = kp.ao[j];
  const int c0 = cd0.x, d0 = cd0.y;
  const int n = w.nao;
  const double* __restrict__ D = w.D;
#pragma unroll
  for (int c = 0; c < NC; ++c)
#pragma unroll
    for (int d = 0; d < ND; ++d) Dcd_s[32 * (c * ND + d)] = D[(long)(c0 + c) * n + d0 + d];
  {  // D_ad of this lane is the same for every row of the block (the rows of a bra half share shell a): once, not per row
    const int a0b = bp.ao[i_first].x;
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
      for (int d = 0; d < ND; ++d) Dad_s[32 * (a * ND + d)] = D[(long)(a0b + a) * n + d0 + d];
  }
  double keepD[6];   // centre D: -(A + B + C), J then K, summed over the rows of this warp
#pragma unroll
  for (int e = 0; e < 6; ++e) keepD[e] = 0.0;
  bool any_row = false;

#pragma unroll 1
  for (int y = gq; y < TILE_ROWS; y += BI) {
    const int i = i_first + y;
    const double qi = bp.q[i];
    if (qi < 0.0 || qi * qk_max < w.thr) break;            // rows are sorted: no later row has work (reading R7)
    const bool active = qj >= 0.0 && qi * qj >= w.thr && (!w.same || j <= i);
    if (!__any_sync(0xffffffffu, active)) continue;
    any_row = true;
    const int2 ab0 = bp.ao[i];
    const int a0 = ab0.x, b0 = ab0.y;
    // ---- density blocks of this row ----
    __syncwarp();
    for (int e = x; e < NA * NB; e += 32) Dab_s[e] = D[(long)(a0 + e / NB) * n + b0 + e % NB];
    for (int e = x & 15; e < NA * NC; e += 16) Dac_s[e] = D[(long)(a0 + e / NC) * n + c0 + e % NC];   // each half stages its own c
    for (int e = x & 15; e < NB * NC; e += 16) Dbc_s[e] = D[(long)(b0 + e / NC) * n + c0 + e % NC];
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
      for (int d = 0; d < ND; ++d) Dbd_s[32 * (b * ND + d)] = D[(long)(b0 + b) * n + d0 + d];
    __syncwarp();
    double acc[18];   // [J: A xyz, B xyz, C xyz | K: same]
#pragma unroll
    for (int e = 0; e < 18; ++e) acc[e] = 0.0;
    if (active) {
      double f = bp.geom[6 * bp.stride + i] * kp.geom[6 * kp.stride + j];
      if (w.same && i == j) f *= 0.5;
      double A[3], AB[3], C[3], CD[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        A[c] = bp.geom[c * bp.stride + i]; AB[c] = bp.geom[(3 + c) * bp.stride + i];
        C[c] = kp.geom[c * kp.stride + j]; CD[c] = kp.geom[(3 + c) * kp.stride + j];
      }
      for (int kb = 0; kb < bp.npp; ++kb) {
        const double p = bp.prim[(kb * 5 + 0) * bp.stride + i];
        const double P[3] = {bp.prim[(kb * 5 + 1) * bp.stride + i], bp.prim[(kb * 5 + 2) * bp.stride + i], bp.prim[(kb * 5 + 3) * bp.stride + i]};
        const double Kab = bp.prim[(kb * 5 + 4) * bp.stride + i];
        const double ea2 = 2.0 * bp.aexp[(kb * 2 + 0) * bp.stride + i], eb2 = 2.0 * bp.aexp[(kb * 2 + 1) * bp.stride + i];
        const double hp = 0.5 / p;
        for (int kk = 0; kk < kp.npp; ++kk) {
          const double q = kp.prim[(kk * 5 + 0) * kp.stride + j];
          const double Q[3] = {kp.prim[(kk * 5 + 1) * kp.stride + j], kp.prim[(kk * 5 + 2) * kp.stride + j], kp.prim[(kk * 5 + 3) * kp.stride + j]};
          const double Kcd = kp.prim[(kk * 5 + 4) * kp.stride + j];
          const double ec2 = 2.0 * kp.aexp[(kk * 2 + 0) * kp.stride + j];
          const double rpq = 1.0 / (p + q), rho = p * q * rpq;
          const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
          const double xx = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
          const double pref = f * Kab * Kcd * sqrt(rpq);
          const double hq = 0.5 / q;
          double u[N], wt[N];
          rys_roots_smem<N>(xx, rtab, w.rys, u, wt);
          if constexpr (MODE == 1) {
#pragma unroll 1
            for (int rt = 0; rt < N; ++rt) {
              const double t2 = u[rt] * rpq;
              const double b00 = 0.5 * t2, b10 = hp - q * t2 * hp, b01 = hq - p * t2 * hq;
              const double c00[3] = {(P[0] - A[0]) - q * t2 * PQ[0], (P[1] - A[1]) - q * t2 * PQ[1], (P[2] - A[2]) - q * t2 * PQ[2]};
              const double c00p[3] = {(Q[0] - C[0]) + p * t2 * PQ[0], (Q[1] - C[1]) + p * t2 * PQ[1], (Q[2] - C[2]) + p * t2 * PQ[2]};
              const double init[3] = {1.0, 1.0, pref * wt[rt]};
              tile_grad_axis<LA, LB, LC, LD, 0>(acc, c00, c00p, init, b10, b01, b00, AB, CD, ea2, eb2, ec2, Dab_s, Dac_s, Dbc_s, Dcd_s, Dad_s, Dbd_s);
              tile_grad_axis<LA, LB, LC, LD, 1>(acc, c00, c00p, init, b10, b01, b00, AB, CD, ea2, eb2, ec2, Dab_s, Dac_s, Dbc_s, Dcd_s, Dad_s, Dbd_s);
              tile_grad_axis<LA, LB, LC, LD, 2>(acc, c00, c00p, init, b10, b01, b00, AB, CD, ea2, eb2, ec2, Dab_s, Dac_s, Dbc_s, Dcd_s, Dad_s, Dbd_s);
            }
          } else {
#pragma unroll
          for (int rt = 0; rt < N; ++rt) {
            const double t2 = u[rt] * rpq;
            const double b00 = 0.5 * t2, b10 = hp - q * t2 * hp, b01 = hq - p * t2 * hq;
            double gx[G2], gy[G2], gz[G2];
            fill_2d_tile<LA + 1, LB + 1, LC + 1, LD>(gx, 1.0, (P[0] - A[0]) - q * t2 * PQ[0], (Q[0] - C[0]) + p * t2 * PQ[0], b10, b01, b00, AB[0], CD[0]);
            fill_2d_tile<LA + 1, LB + 1, LC + 1, LD>(gy, 1.0, (P[1] - A[1]) - q * t2 * PQ[1], (Q[1] - C[1]) + p * t2 * PQ[1], b10, b01, b00, AB[1], CD[1]);
            fill_2d_tile<LA + 1, LB + 1, LC + 1, LD>(gz, pref * wt[rt], (P[2] - A[2]) - q * t2 * PQ[2], (Q[2] - C[2]) + p * t2 * PQ[2], b10, b01, b00, AB[2], CD[2]);
            int a = 0;
#pragma unroll
            for (int ax = LA; ax >= 0; --ax)
#pragma unroll
            for (int ay = LA - ax; ay >= 0; --ay) {
              const int az = LA - ax - ay;
              int b = 0;
#pragma unroll
              for (int bx = LB; bx >= 0; --bx)
#pragma unroll
              for (int by = LB - bx; by >= 0; --by) {
                const int bz = LB - bx - by;
                const double dab = Dab_s[a * NB + b];
                int c = 0;
#pragma unroll
                for (int cx = LC; cx >= 0; --cx)
#pragma unroll
                for (int cy = LC - cx; cy >= 0; --cy) {
                  const int cz = LC - cx - cy;
                  const double dac = Dac_s[a * NC + c], dbc = Dbc_s[b * NC + c];
                  int d = 0;
#pragma unroll
                  for (int dx = LD; dx >= 0; --dx)
#pragma unroll
                  for (int dy = LD - dx; dy >= 0; --dy) {
                    const int dz = LD - dx - dy;
                    const double pj = dab * Dcd_s[32 * (c * ND + d)];
                    const double pk = fma(dac, Dbd_s[32 * (b * ND + d)], Dad_s[32 * (a * ND + d)] * dbc);
                    const int ex = ax * SA + bx * SB + cx * SC + dx * SD;
                    const int ey = ay * SA + by * SB + cy * SC + dy * SD;
                    const int ez = az * SA + bz * SB + cz * SC + dz * SD;
                    const double vx = gx[ex], vy = gy[ey], vz = gz[ez];
                    const double oyz = vy * vz, oxz = vx * vz, oxy = vx * vy;
                    // F[I](i) = 2 alpha I(i+1) - i I(i-1) on the differentiated centre and axis (Eq. 11)
                    const double dAx = ax > 0 ? fma(ea2, gx[ex + SA], -ax * gx[ex - SA]) : ea2 * gx[ex + SA];
                    const double dAy = ay > 0 ? fma(ea2, gy[ey + SA], -ay * gy[ey - SA]) : ea2 * gy[ey + SA];
                    const double dAz = az > 0 ? fma(ea2, gz[ez + SA], -az * gz[ez - SA]) : ea2 * gz[ez + SA];
                    const double dBx = bx > 0 ? fma(eb2, gx[ex + SB], -bx * gx[ex - SB]) : eb2 * gx[ex + SB];
                    const double dBy = by > 0 ? fma(eb2, gy[ey + SB], -by * gy[ey - SB]) : eb2 * gy[ey + SB];
                    const double dBz = bz > 0 ? fma(eb2, gz[ez + SB], -bz * gz[ez - SB]) : eb2 * gz[ez + SB];
                    const double dCx = cx > 0 ? fma(ec2, gx[ex + SC], -cx * gx[ex - SC]) : ec2 * gx[ex + SC];
                    const double dCy = cy > 0 ? fma(ec2, gy[ey + SC], -cy * gy[ey - SC]) : ec2 * gy[ey + SC];
                    const double dCz = cz > 0 ? fma(ec2, gz[ez + SC], -cz * gz[ez - SC]) : ec2 * gz[ez + SC];
                    const double jx = pj * oyz, jy = pj * oxz, jz = pj * oxy;
                    const double kx = pk * oyz, ky = pk * oxz, kz = pk * oxy;
                    acc[0] = fma(dAx, jx, acc[0]); acc[1] = fma(dAy, jy, acc[1]); acc[2] = fma(dAz, jz, acc[2]);
                    acc[3] = fma(dBx, jx, acc[3]); acc[4] = fma(dBy, jy, acc[4]); acc[5] = fma(dBz, jz, acc[5]);
                    acc[6] = fma(dCx, jx, acc[6]); acc[7] = fma(dCy, jy, acc[7]); acc[8] = fma(dCz, jz, acc[8]);
                    acc[9] = fma(dAx, kx, acc[9]); acc[10] = fma(dAy, ky, acc[10]); acc[11] = fma(dAz, kz, acc[11]);
                    acc[12] = fma(dBx, kx, acc[12]); acc[13] = fma(dBy, ky, acc[13]); acc[14] = fma(dBz, kz, acc[14]);
                    acc[15] = fma(dCx, kx, acc[15]); acc[16] = fma(dCy, ky, acc[16]); acc[17] = fma(dCz, kz, acc[17]);
                    ++d;
                  }
                  ++c;
                }
                ++b;
              }
              ++a;
            }
          }
          }
        }
      }
#pragma unroll
      for (int e = 0; e < 9; ++e) { acc[e] *= 4.0; acc[9 + e] *= 2.0; }   // PJ = 4 f ..., PK = 2 f ... (f is in pref)
#pragma unroll
      for (int ax = 0; ax < 3; ++ax) {
        keepD[ax] -= acc[ax] + acc[3 + ax] + acc[6 + ax];
        keepD[3 + ax] -= acc[9 + ax] + acc[12 + ax] + acc[15 + ax];
      }
    }
    // centres A, B (fixed for the row) and C (shared by the lanes): sum over the lanes, 18 atomics per row
    const int2 at_ab = bp.atom[i];
    const int atC_lo = kp.atom[j_first].x, atC_hi = kp.atom[j_first + 16].x;   // the two ket halves have their own shell c
    warp_reduce_values<18, true>(acc, stage, x, [&](int v, int half, double sum) {
      const int jk = v / 9, ce = (v % 9) / 3, ax = v % 3;
      const int at = ce == 0 ? at_ab.x : ce == 1 ? at_ab.y : half ? atC_hi : atC_lo;
      atomic_add((jk ? w.gK : w.gJ) + 3 * at + ax, sum);
    });
  }
  if (any_row) {
    const int atD = kp.atom[j].y;
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
      if (keepD[ax] != 0.0) atomic_add(w.gJ + 3 * atD + ax, keepD[ax]);
      if (keepD[3 + ax] != 0.0) atomic_add(w.gK + 3 * atD + ax, keepD[3 + ax]);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// MODE 2, "axis team": the classes from 27 Cartesian elements on.  With one thread per quartet the density products
// pj = D_ab D_cd, pk = D_ac D_bd + D_ad D_bc of all elements are loop invariants that the compiler keeps live across the
// three axis passes; beside the 2-D integrals they do not fit the register file and spilled (profiles/r02_cfg4.md:
// tile_grad_kernel<2,1,1,0>: 65 % of the stall samples wait on local-memory loads, 15 GB of DRAM writes per launch).
// Here a quartet belongs to a TEAM of three threads at the same lane of three warps; thread t owns the differentiated
// axis t: it builds the 2-D integrals of axis t raised and of the other two plain -- exactly one axis pass of MODE 1, so
// the team does no arithmetic twice -- and accumulates its 6 scalars (centres A, B, C x {J, K}).  pj and pk are formed
// once per row by the team (a third of the elements each) in a shared-memory column per lane and read back with two
// conflict-free loads per element and root; two named barriers per row keep the team in step.
template <int LA, int LB, int LC, int LD, int BI>
struct TileGradTeamTraits {
  static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD), NE = NA * NB * NC * ND;
  static constexpr int N = nroots_of(LA + LB + LC + LD + 1);
  static constexpr int NUNI = NA * NB + 2 * (NA * NC + NB * NC);
  static constexpr int NLANE = NC * ND + NA * ND + NB * ND;
  static constexpr int STAGE = reduce_stage_size(6);                  // per warp
  static constexpr int PERTEAM = 3 * STAGE + NUNI + 32 * NLANE + 2 * NE * 32;
  static constexpr int RT = rys2_size(N);
  static constexpr size_t SMEM = sizeof(double) * (RT + BI * PERTEAM);
};

template <int LA, int LB, int LC, int LD, int BI>
__global__ void __launch_bounds__(96 * BI) tile_grad_team_kernel(Work w) {
  using Tr = TileGradTeamTraits<LA, LB, LC, LD, BI>;
  constexpr int NA = Tr::NA, NB = Tr::NB, NC = Tr::NC, ND = Tr::ND, NE = Tr::NE, N = Tr::N;
  extern __shared__ __align__(16) double smem[];

  const PairSet& bp = w.bra; const PairSet& kp = w.ket;
  const int blk = blockIdx.x * w.nshard + w.shard;
  if (blk >= w.row_off[w.nrows]) return;
  const int r = find_row_warp(w.row_off, w.nrows, blk, threadIdx.x);
  const int x = threadIdx.x, wy = threadIdx.y, gq = wy / 3, t = wy - 3 * gq;   // team gq, differentiated axis t
  const int i_first = w.row_slot[r], j_first = (blk - w.row_off[r]) * 32;
  const double* rtab = smem;
  rys_stage_table<N>(smem, w.rys, wy * 32 + x, 96 * BI);
  __syncthreads();
  double* team = smem + Tr::RT + gq * Tr::PERTEAM;
  double* stage = team + t * Tr::STAGE;             // warp-private reduction staging
  double* uni = team + 3 * Tr::STAGE;               // [D_ab | D_ac | D_bc] (per ket half), the same for all lanes
  double* mine = uni + Tr::NUNI + x;                // column of this lane, stride 32: [D_cd | D_ad | D_bd]
  double* pjk = uni + Tr::NUNI + 32 * Tr::NLANE + x;   // column of this lane: pj[e] at 32 e, pk[e] at 32 (NE + e)
  const int half = x >> 4;
  double* Dab_s = uni; double* Dac_s = uni + NA * NB + half * (NA * NC + NB * NC); double* Dbc_s = Dac_s + NA * NC;
  double* Dcd_s = mine; double* Dad_s = mine + 32 * NC * ND; double* Dbd_s = Dad_s + 32 * NA * ND;
  const int bar_id = 1 + gq;                        // named barrier of the team (barrier 0 is __syncthreads)

  const int j = j_first + x;
  const double qj = kp.q[j];
  double qk_max = qj;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) qk_max = fmax(qk_max, __shfl_xor_sync(0xffffffffu, qk_max, o));
  const int2 cd0 = kp.ao[j];
  const int c0 = cd0.x, d0 = cd0.y;
  const int n = w.nao;
  const double* __restrict__ D = w.D;
  if (t == 0) {
#pragma unroll
    for (int c = 0; c < NC; ++c)
#pragma unroll
      for (int d = 0; d < ND; ++d) Dcd_s[32 * (c * ND + d)] = D[(long)(c0 + c) * n + d0 + d];
  }
  if (t == 1) {   // D_ad of this lane: the same for every row of the block (the first row's barrier publishes it to the team)
    const int a0b = bp.ao[i_first].x;
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
      for (int d = 0; d < ND; ++d) Dad_s[32 * (a * ND + d)] = D[(long)(a0b + a) * n + d0 + d];
  }
  double keepD[2] = {0.0, 0.0};   // centre D of this thread's axis: -(A + B + C), J and K, over the rows
  bool any_row = false;

#pragma unroll 1
  for (int y = gq; y < TILE_ROWS; y += BI) {
    const int i = i_first + y;
    const double qi = bp.q[i];
    if (qi < 0.0 || qi * qk_max < w.thr) break;            // the same decision in the three warps of the team
    const bool active = qj >= 0.0 && qi * qj >= w.thr && (!w.same || j <= i);
    if (!__any_sync(0xffffffffu, active)) continue;
    any_row = true;
    const int2 ab0 = bp.ao[i];
    const int a0 = ab0.x, b0 = ab0.y;
    // ---- density blocks of this row: the three warps of the team share the work ----
    if (t == 0) {
      for (int e = x; e < NA * NB; e += 32) Dab_s[e] = D[(long)(a0 + e / NB) * n + b0 + e % NB];
      for (int e = x & 15; e < NA * NC; e += 16) Dac_s[e] = D[(long)(a0 + e / NC) * n + c0 + e % NC];
      for (int e = x & 15; e < NB * NC; e += 16) Dbc_s[e] = D[(long)(b0 + e / NC) * n + c0 + e % NC];
    } else if (t == 2) {
#pragma unroll
      for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int d = 0; d < ND; ++d) Dbd_s[32 * (b * ND + d)] = D[(long)(b0 + b) * n + d0 + d];
    }
    asm volatile("bar.sync %0, 96;" ::"r"(bar_id) : "memory");
    // pj, pk of the elements e = t, t + 3, ... (run-time element index: this loop is short and not unrolled)
#pragma unroll 1
    for (int e = t; e < NE; e += 3) {
      const int d = e % ND, t1 = e / ND, c = t1 % NC, t2 = t1 / NC, b = t2 % NB, a = t2 / NB;
      pjk[32 * e] = Dab_s[a * NB + b] * Dcd_s[32 * (c * ND + d)];
      pjk[32 * (NE + e)] = fma(Dac_s[a * NC + c], Dbd_s[32 * (b * ND + d)], Dad_s[32 * (a * ND + d)] * Dbc_s[b * NC + c]);
    }
    asm volatile("bar.sync %0, 96;" ::"r"(bar_id) : "memory");

    double acc[6];   // [J: A, B, C | K: A, B, C] of axis t
#pragma unroll
    for (int e = 0; e < 6; ++e) acc[e] = 0.0;
    if (active) {
      double f = bp.geom[6 * bp.stride + i] * kp.geom[6 * kp.stride + j];
      if (w.same && i == j) f *= 0.5;
      double A[3], AB[3], C[3], CD[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        A[c] = bp.geom[c * bp.stride + i]; AB[c] = bp.geom[(3 + c) * bp.stride + i];
        C[c] = kp.geom[c * kp.stride + j]; CD[c] = kp.geom[(3 + c) * kp.stride + j];
      }
      for (int kb = 0; kb < bp.npp; ++kb) {
        const double p = bp.prim[(kb * 5 + 0) * bp.stride + i];
        const double P[3] = {bp.prim[(kb * 5 + 1) * bp.stride + i], bp.prim[(kb * 5 + 2) * bp.stride + i], bp.prim[(kb * 5 + 3) * bp.stride + i]};
        const double Kab = bp.prim[(kb * 5 + 4) * bp.stride + i];
        const double ea2 = 2.0 * bp.aexp[(kb * 2 + 0) * bp.stride + i], eb2 = 2.0 * bp.aexp[(kb * 2 + 1) * bp.stride + i];
        const double hp = 0.5 / p;
        for (int kk = 0; kk < kp.npp; ++kk) {
          const double q = kp.prim[(kk * 5 + 0) * kp.stride + j];
          const double Q[3] = {kp.prim[(kk * 5 + 1) * kp.stride + j], kp.prim[(kk * 5 + 2) * kp.stride + j], kp.prim[(kk * 5 + 3) * kp.stride + j]};
          const double Kcd = kp.prim[(kk * 5 + 4) * kp.stride + j];
          const double ec2 = 2.0 * kp.aexp[(kk * 2 + 0) * kp.stride + j];
          const double rpq = 1.0 / (p + q), rho = p * q * rpq;
          const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
          const double xx = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
          const double pref = f * Kab * Kcd * sqrt(rpq);
          const double hq = 0.5 / q;
          double u[N], wt[N];
          rys_roots_smem<N>(xx, rtab, w.rys, u, wt);
#pragma unroll 1
          for (int rt = 0; rt < N; ++rt) {
            const double t2 = u[rt] * rpq;
            const double b00 = 0.5 * t2, b10 = hp - q * t2 * hp, b01 = hq - p * t2 * hq;
            const double c00[3] = {(P[0] - A[0]) - q * t2 * PQ[0], (P[1] - A[1]) - q * t2 * PQ[1], (P[2] - A[2]) - q * t2 * PQ[2]};
            const double c00p[3] = {(Q[0] - C[0]) + p * t2 * PQ[0], (Q[1] - C[1]) + p * t2 * PQ[1], (Q[2] - C[2]) + p * t2 * PQ[2]};
            const double init[3] = {1.0, 1.0, pref * wt[rt]};
            switch (t) {   // warp-uniform: team members are warps
              case 0: tile_grad_team_axis<LA, LB, LC, LD, 0>(acc, c00, c00p, init, b10, b01, b00, AB, CD, ea2, eb2, ec2, pjk); break;
              case 1: tile_grad_team_axis<LA, LB, LC, LD, 1>(acc, c00, c00p, init, b10, b01, b00, AB, CD, ea2, eb2, ec2, pjk); break;
              default: tile_grad_team_axis<LA, LB, LC, LD, 2>(acc, c00, c00p, init, b10, b01, b00, AB, CD, ea2, eb2, ec2, pjk); break;
            }
          }
        }
      }
#pragma unroll
      for (int e = 0; e < 3; ++e) { acc[e] *= 4.0; acc[3 + e] *= 2.0; }   // PJ = 4 f ..., PK = 2 f ... (f is in pref)
      keepD[0] -= acc[0] + acc[1] + acc[2];
      keepD[1] -= acc[3] + acc[4] + acc[5];
    }
    const int2 at_ab = bp.atom[i];
    const int atC_lo = kp.atom[j_first].x, atC_hi = kp.atom[j_first + 16].x;
    warp_reduce_values<6, true>(acc, stage, x, [&](int v, int hf, double sum) {
      const int jk = v / 3, ce = v % 3;
      const int at = ce == 0 ? at_ab.x : ce == 1 ? at_ab.y : hf ? atC_hi : atC_lo;
      atomic_add((jk ? w.gK : w.gJ) + 3 * at + t, sum);
    });
  }
  if (any_row) {
    const int atD = kp.atom[j].y;
    if (keepD[0] != 0.0) atomic_add(w.gJ + 3 * atD + t, keepD[0]);
    if (keepD[1] != 0.0) atomic_add(w.gK + 3 * atD + t, keepD[1]);
  }
}

template <int LA, int LB, int LC, int LD, int BI, int MODE>
cudaError_t launch_tile_grad(const Work& w, int nblocks_dense, cudaStream_t s) {
  const int grid = (nblocks_dense + w.nshard - 1) / w.nshard;
  if (grid <= 0) return cudaSuccess;
  static bool attr_set = false;
  if constexpr (MODE == 2) {
    using Tr = TileGradTeamTraits<LA, LB, LC, LD, BI>;
    static_assert(Tr::SMEM <= 227 * 1024, "axis-team gradient kernel: shared memory");
    if (!attr_set) {
      cudaError_t e = cudaFuncSetAttribute(tile_grad_team_kernel<LA, LB, LC, LD, BI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tr::SMEM);
      if (e != cudaSuccess) return e;
      attr_set = true;
    }
    tile_grad_team_kernel<LA, LB, LC, LD, BI><<<grid, dim3(32, 3 * BI), Tr::SMEM, s>>>(w);
  } else {
    using Tr = TileGradTraits<LA, LB, LC, LD, BI, MODE>;
    static_assert(Tr::SMEM <= 227 * 1024, "tile gradient kernel: shared memory");
    if (!attr_set) {
      cudaError_t e = cudaFuncSetAttribute(tile_grad_kernel<LA, LB, LC, LD, BI, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tr::SMEM);
      if (e != cudaSuccess) return e;
      attr_set = true;
    }
    tile_grad_kernel<LA, LB, LC, LD, BI, MODE><<<grid, dim3(32, BI), Tr::SMEM, s>>>(w);
  }
  return cudaGetLastError();
}

}  // namespace eri
