// tile_kernel.cuh -- tile family of J/K kernels (family T).
// The paper's Algorithm 2 keeps the 2-D integrals of one root and the contracted block of a
// quartet in registers and then issues six FP64 atomics PER ELEMENT.  On sm_100a a
// scattered FP64 reduction costs more SM time than the arithmetic of a low-l quartet, so this family keeps the
// register-resident evaluation and changes everything around it:
//   * pairs are laid out in HALF-CHUNKS of 16 slots that share their first shell and are sorted by decreasing Schwarz
//     factor (api.cu, "grouped pair sets"); a block is (one bra half: 16 rows, one shell a) x (one ket chunk: two halves
//     = the 32 lanes of a warp, one shell c per half).  A warp takes one bra row at a time (lane = ket slot) and skips
//     the rows that Schwarz rules out;
//   * a quartet is evaluated by TQ threads that sit in TQ different warps (same lane): each owns NA/TQ Cartesian
//     components of shell a and recomputes the (cheap) 2-D integrals, so that its accumulators fit in registers and
//     no warp ever diverges;
//   * contract, then digest once per quartet into six small per-thread blocks.  J_cd and K_ad (targets fixed per lane
//     while the warp walks down the rows) are kept in shared memory until the block ends; J_ab, K_ac, K_bc
//     (targets fixed per row) are summed over the lanes through a warp-private shared-memory transpose; only K_bd is
//     private to a quartet.  One block barrier, at the end.  FP64 atomics leave once per tile edge element.
// The horizontal transfer is built on the first centre of each pair; the host only selects this family when that is
// numerically safe for every pair of the unit (api.cu, "hrr_loss").
#pragma once
#include "eri_dev.cuh"
#include "launch.h"

namespace eri {

constexpr int TILE_ROWS = 16;   // bra slots per half-chunk = rows of a block's tile (they share the first shell a)

// 2-D integrals of one axis and one root in registers: G[((i*(LB+1)+j)*(LC+1)+k)*(LD+1)+l] (reading R5).
template <int LA, int LB, int LC, int LD>
__device__ __forceinline__ void fill_2d_tile(double* __restrict__ G, double init, double c00, double c00p, double b10,
                                             double b01, double b00, double x12, double x34) {
  constexpr int NM = LA + LB, MM = LC + LD;
  constexpr int SL = 1, SK = LD + 1, SJ = (LC + 1) * SK, SI = (LB + 1) * SJ;
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
  for (int j = 0; j <= LB; ++j) {
    if (j > 0) {
#pragma unroll
      for (int i = 0; i <= NM - j; ++i)
#pragma unroll
        for (int m = 0; m <= MM; ++m) T[i][m] = fma(x12, T[i][m], T[i + 1][m]);
    }
#pragma unroll
    for (int i = 0; i <= LA; ++i) {
      double R[MM + 1];
#pragma unroll
      for (int m = 0; m <= MM; ++m) R[m] = T[i][m];
#pragma unroll
      for (int l = 0; l <= LD; ++l) {
        if (l > 0) {
#pragma unroll
          for (int k = 0; k <= MM - l; ++k) R[k] = fma(x34, R[k], R[k + 1]);
        }
#pragma unroll
        for (int k = 0; k <= LC; ++k) G[i * SI + j * SJ + k * SK + l * SL] = R[k];
      }
    }
  }
}

// g[(ai*NB + b)*NCD + c*ND + d] += X Y Z for the components a = T*NAT + ai owned by team member T (Eq. 1)
template <int LA, int LB, int LC, int LD, int NAT, int T>
__device__ __forceinline__ void tile_product(double* __restrict__ g, const double* __restrict__ gx,
                                             const double* __restrict__ gy, const double* __restrict__ gz) {
  constexpr int NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
  constexpr int SC = LD + 1, SB = (LC + 1) * SC, SA = (LB + 1) * SB;
  int a = 0;
#pragma unroll
  for (int ax = LA; ax >= 0; --ax)
#pragma unroll
  for (int ay = LA - ax; ay >= 0; --ay) {
    if (a >= T * NAT && a < (T + 1) * NAT) {
      const int az = LA - ax - ay, ai = a - T * NAT;
      int b = 0;
#pragma unroll
      for (int bx = LB; bx >= 0; --bx)
#pragma unroll
      for (int by = LB - bx; by >= 0; --by) {
        const int bz = LB - bx - by;
        int c = 0;
#pragma unroll
        for (int cx = LC; cx >= 0; --cx)
#pragma unroll
        for (int cy = LC - cx; cy >= 0; --cy) {
          const int cz = LC - cx - cy;
          int d = 0;
#pragma unroll
          for (int dx = LD; dx >= 0; --dx)
#pragma unroll
          for (int dy = LD - dx; dy >= 0; --dy) {
            const int dz = LD - dx - dy;
            const int e = ((ai * NB + b) * NC + c) * ND + d;
            g[e] = fma(gx[ax * SA + bx * SB + cx * SC + dx] * gy[ay * SA + by * SB + cy * SC + dy],
                       gz[az * SA + bz * SB + cz * SC + dz], g[e]);
            ++d;
          }
          ++c;
        }
        ++b;
      }
    }
    ++a;
  }
}

// Sum of NV per-lane values over the lanes of a warp: lanes stage their values in the warp's private region
// stage[32][33] (value-row major, 32 values per batch) and lane l adds up value-row l.  HALVES = false: one sum over the
// 32 lanes, emit(v, 0, sum).  HALVES = true: lanes 0-15 and 16-31 belong to two half-chunks of the ket set (different
// first shells c), so the two halves are summed separately, emit(v, half, sum).
template <int NV, bool HALVES, class F>
__device__ __forceinline__ void warp_reduce_values(const double* __restrict__ v, double* __restrict__ stage, int lane, F emit) {
  if constexpr (NV <= 16) {
    // few values: all 32 lanes work.  ROWS value-rows x LPR lanes per row; a lane adds ROWS staged elements of its row
    // (within its ket half if HALVES), then the LPR (LPR/2) lanes of a row (half) finish with shuffles.
    constexpr int ROWS = NV <= 1 ? 1 : NV <= 2 ? 2 : NV <= 4 ? 4 : NV <= 8 ? 8 : 16;
    constexpr int LPR = 32 / ROWS, GRP = HALVES ? LPR / 2 : LPR;   // lanes per row; lanes that share one sum
    constexpr int RS = 32 + LPR;                                    // row stride: lane id == bank (mod 16) on both sides
    // staged position of the value of source lane L: the elements of ket half h land on the columns that the lanes of
    // half h read (column mod LPR in [h GRP, (h+1) GRP)), so that lane sl of a row simply reads columns sl + m LPR
    const int q = lane & 15, hl = lane >> 4;
    const int pos = HALVES ? (q / GRP) * LPR + hl * GRP + (q % GRP) : lane;
    __syncwarp();
#pragma unroll
    for (int i = 0; i < NV; ++i) stage[i * RS + pos] = v[i];
    __syncwarp();
    const int row = lane / LPR, sl = lane - row * LPR;
    const int half = HALVES ? sl / GRP : 0, t = sl - half * GRP;
    const double* src = stage + row * RS + sl;
    double sum = 0.0;
#pragma unroll
    for (int m = 0; m < ROWS; ++m) sum += src[m * LPR];
#pragma unroll
    for (int o = GRP / 2; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    if (t == 0 && row < NV && sum != 0.0) emit(row, half, sum);
  } else {
#pragma unroll
    for (int b0 = 0; b0 < NV; b0 += 32) {
      const int nb = NV - b0 < 32 ? NV - b0 : 32;
      __syncwarp();
#pragma unroll
      for (int i = 0; i < 32; ++i) if (i < nb) stage[i * 33 + lane] = v[b0 + i];
      __syncwarp();
      if (lane < nb) {
        const double* row = stage + lane * 33;
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
        for (int k = 0; k < 16; k += 2) { s0 += row[k]; s1 += row[k + 1]; s2 += row[16 + k]; s3 += row[17 + k]; }
        if (HALVES) {
          const double lo = s0 + s1, hi = s2 + s3;
          if (lo != 0.0) emit(b0 + lane, 0, lo);
          if (hi != 0.0) emit(b0 + lane, 1, hi);
        } else {
          const double sum = (s0 + s1) + (s2 + s3);
          if (sum != 0.0) emit(b0 + lane, 0, sum);
        }
      }
    }
  }
}

// doubles of warp-private staging that warp_reduce_values<NV> touches
__host__ __device__ constexpr int reduce_stage_size(int nv) {
  if (nv > 16) return 32 * 33;
  const int rows = nv <= 1 ? 1 : nv <= 2 ? 2 : nv <= 4 ? 4 : nv <= 8 ? 8 : 16;
  return rows * (32 + 32 / rows);
}
__host__ __device__ constexpr int max3(int a, int b, int c) { return a > b ? (a > c ? a : c) : (b > c ? b : c); }

template <int LA, int LB, int LC, int LD, int TQ, int BI>
struct TileTraits {
  static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
  static_assert(NA % TQ == 0, "TQ must divide the number of Cartesian components of shell a");
  static constexpr int NAT = NA / TQ, NABT = NAT * NB, NCD = NC * ND, NE = NABT * NCD;
  static constexpr int N = nroots_of(LA + LB + LC + LD);
  static constexpr int G2 = (LA + 1) * (LB + 1) * (LC + 1) * (LD + 1);
  static constexpr int NW = BI * TQ, NT = 32 * NW;          // BI = quartet warps per block
  // blocks per SM asked of the compiler (0 = unspecified), by block size and register demand RW = accumulators + 2-D integrals of
  // one root; fitted to per-class timings on cfg3: more resident warps pay off until the tighter register cap makes the kernel spill
  static constexpr int RW = NE + 3 * G2;
  static constexpr int MINB = (NT == 128 && RW <= 63) ? 3 : (NT == 256 && TQ == 1 && RW >= 30) ? 2 : (NT == 256 && RW <= 15) ? 4 : 0;
  static constexpr int NKEEP = NCD + NAT * ND;              // per-thread sums kept over the rows: J_cd, K_ad
  static constexpr int STAGE = max3(reduce_stage_size(NABT), reduce_stage_size(NAT * NC), reduce_stage_size(NB * NC));   // doubles per warp
  static constexpr int RT = rys2_size(N);                    // the class's Rys table, first in the block's shared memory (16-byte aligned)
  static constexpr size_t SMEM = sizeof(double) * (RT + NW * STAGE + 2 * NKEEP * NT);   // + D_cd, D_ad of every thread, fixed for the block
};

template <int LA, int LB, int LC, int LD, int TQ, int BI>
__global__ void __launch_bounds__(32 * BI * TQ, (TileTraits<LA, LB, LC, LD, TQ, BI>::MINB)) tile_jk_kernel(Work w) {
  using Tr = TileTraits<LA, LB, LC, LD, TQ, BI>;
  constexpr int NB = Tr::NB, NC = Tr::NC, ND = Tr::ND, NAT = Tr::NAT, NABT = Tr::NABT, NCD = Tr::NCD, NE = Tr::NE;
  constexpr int N = Tr::N, G2 = Tr::G2, NT = Tr::NT, NKEEP = Tr::NKEEP;
  extern __shared__ __align__(16) double smem[];

  const PairSet& bp = w.bra; const PairSet& kp = w.ket;
  const int blk = blockIdx.x * w.nshard + w.shard;
  if (blk >= w.row_off[w.nrows]) return;
  const int r = find_row_warp(w.row_off, w.nrows, blk, threadIdx.x);
  const int x = threadIdx.x, wy = threadIdx.y, gq = wy / TQ, t = wy - gq * TQ, tid = wy * 32 + x;
  const int i_first = w.row_slot[r], j_first = (blk - w.row_off[r]) * 32;
  const double* rtab = smem;                        // Rys table of the class (eri_dev.cuh "Shared-memory copy")
  rys_stage_table<N>(smem, w.rys, tid, NT);
  double* stage = smem + Tr::RT + wy * Tr::STAGE;
  double* keep = smem + Tr::RT + Tr::NW * Tr::STAGE + tid;   // keep[e * NT]: [0, NCD) J_cd ; [NCD, NCD + NAT*ND) K_ad
  const double* hold = keep + NKEEP * NT;                    // hold[e * NT]: [0, NCD) D_cd ; [NCD, NCD + NAT*ND) D_ad (filled below)
#pragma unroll
  for (int e = 0; e < NKEEP; ++e) keep[e * NT] = 0.0;
  __syncthreads();

  // ---- this lane's ket pair (fixed for the whole block) ----
  const int j = j_first + x;
  const double qj = kp.q[j];
  double qk_max = qj;   // largest Schwarz factor of the ket chunk
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) qk_max = fmax(qk_max, __shfl_xor_sync(0xffffffffu, qk_max, o));
  const int2 cd0 = kp.ao[j];
  const int c0 = cd0.x, d0 = cd0.y;
  const int c0_lo = __shfl_sync(0xffffffffu, c0, 0), c0_hi = __shfl_sync(0xffffffffu, c0, 16);   // shell c of the two ket halves
  const int n = w.nao;
  const double* __restrict__ D = w.D;
  double* __restrict__ Jm = w.J; double* __restrict__ Km = w.K;
  // The density blocks D_cd and D_ad of this thread do not change from row to row (its ket pair is fixed, and the rows of a bra
  // half share shell a): read once per block.  Per row they were NCD + NAT ND loads whose 32 lanes hit 20-30 different cache
  // lines each -- a third of the global tag requests of the (ps|ss) kernel (profiles/r02_cfg3.md section 6).
  {
    double* hw = keep + NKEEP * NT;
    const int a0b = bp.ao[i_first].x + t * NAT;
#pragma unroll
    for (int c = 0; c < NC; ++c)
#pragma unroll
      for (int d = 0; d < ND; ++d) hw[(c * ND + d) * NT] = D[(long)(c0 + c) * n + d0 + d];
#pragma unroll
    for (int a = 0; a < NAT; ++a)
#pragma unroll
      for (int d = 0; d < ND; ++d) hw[(NCD + a * ND + d) * NT] = D[(long)(a0b + a) * n + d0 + d];
  }
  int a0 = -1;                         // first Cartesian AO of shell a owned by this thread
  const double thr = w.thr_dev ? *w.thr_dev : w.thr;   // density-weighted call: tau / P_{ab|cd} of this unit (Eq. 8-9)

#pragma unroll 1
  for (int y = gq; y < TILE_ROWS; y += BI) {
    const int i = i_first + y;
    const double qi = bp.q[i];
    if (qi < 0.0 || qi * qk_max < thr) break;              // rows are sorted: no later row has work (reading R7)
    const bool active = qj >= 0.0 && qi * qj >= thr && (!w.same || j <= i);
    if (!__any_sync(0xffffffffu, active)) continue;
    const int2 ab0 = bp.ao[i];
    a0 = ab0.x + t * NAT;
    const int b0 = ab0.y;

    double g[NE];
#pragma unroll
    for (int e = 0; e < NE; ++e) g[e] = 0.0;
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
        const double hp = 0.5 / p;
        for (int kk = 0; kk < kp.npp; ++kk) {
          const double q = kp.prim[(kk * 5 + 0) * kp.stride + j];
          const double Q[3] = {kp.prim[(kk * 5 + 1) * kp.stride + j], kp.prim[(kk * 5 + 2) * kp.stride + j], kp.prim[(kk * 5 + 3) * kp.stride + j]};
          const double Kcd = kp.prim[(kk * 5 + 4) * kp.stride + j];
          const double rpq = 1.0 / (p + q), rho = p * q * rpq;
          const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
          const double xx = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
          const double pref = f * Kab * Kcd * sqrt(rpq);
          const double hq = 0.5 / q;
          double u[N], wt[N];
          rys_roots_smem<N>(xx, rtab, w.rys, u, wt);
#pragma unroll
          for (int rt = 0; rt < N; ++rt) {
            const double t2 = u[rt] * rpq;
            const double b00 = 0.5 * t2, b10 = hp - q * t2 * hp, b01 = hq - p * t2 * hq;
            double gx[G2], gy[G2], gz[G2];
            fill_2d_tile<LA, LB, LC, LD>(gx, 1.0, (P[0] - A[0]) - q * t2 * PQ[0], (Q[0] - C[0]) + p * t2 * PQ[0], b10, b01, b00, AB[0], CD[0]);
            fill_2d_tile<LA, LB, LC, LD>(gy, 1.0, (P[1] - A[1]) - q * t2 * PQ[1], (Q[1] - C[1]) + p * t2 * PQ[1], b10, b01, b00, AB[1], CD[1]);
            fill_2d_tile<LA, LB, LC, LD>(gz, pref * wt[rt], (P[2] - A[2]) - q * t2 * PQ[2], (Q[2] - C[2]) + p * t2 * PQ[2], b10, b01, b00, AB[2], CD[2]);
            if (TQ == 1) tile_product<LA, LB, LC, LD, NAT, 0>(g, gx, gy, gz);
            else {
              switch (t) {   // warp-uniform: team members are warps
                case 0: tile_product<LA, LB, LC, LD, NAT, 0>(g, gx, gy, gz); break;
                case 1: tile_product<LA, LB, LC, LD, NAT, (TQ > 1 ? 1 : 0)>(g, gx, gy, gz); break;
                case 2: tile_product<LA, LB, LC, LD, NAT, (TQ > 2 ? 2 : 0)>(g, gx, gy, gz); break;
                case 3: tile_product<LA, LB, LC, LD, NAT, (TQ > 3 ? 3 : 0)>(g, gx, gy, gz); break;
                case 4: tile_product<LA, LB, LC, LD, NAT, (TQ > 4 ? 4 : 0)>(g, gx, gy, gz); break;
                default: tile_product<LA, LB, LC, LD, NAT, (TQ > 5 ? 5 : 0)>(g, gx, gy, gz); break;
              }
            }
          }
        }
      }
    }

    // ---- digestion: the six updates of Alg. 2 lines 8-13; g = 0 on idle lanes ----
    {  // J_ab += sum_cd g D_cd ; summed over the lanes
      double Dcd[NCD];
#pragma unroll
      for (int c = 0; c < NC; ++c)
#pragma unroll
        for (int d = 0; d < ND; ++d) Dcd[c * ND + d] = hold[(c * ND + d) * NT];
      double v[NABT];
#pragma unroll
      for (int ab = 0; ab < NABT; ++ab) {
        double sacc = 0.0;
#pragma unroll
        for (int cd = 0; cd < NCD; ++cd) sacc = fma(g[ab * NCD + cd], Dcd[cd], sacc);
        v[ab] = sacc;
      }
      warp_reduce_values<NABT, false>(v, stage, x, [&](int vi, int, double sum) { atomic_add(Jm + (long)(a0 + vi / NB) * n + b0 + vi % NB, sum); });
    }
    {  // J_cd += sum_ab g D_ab ; kept per lane over the rows.  D_ab is the same for all lanes (broadcast loads)
      double v[NCD];
#pragma unroll
      for (int cd = 0; cd < NCD; ++cd) v[cd] = 0.0;
#pragma unroll
      for (int a = 0; a < NAT; ++a)
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          const double dab = D[(long)(a0 + a) * n + b0 + b];
#pragma unroll
          for (int cd = 0; cd < NCD; ++cd) v[cd] = fma(g[(a * NB + b) * NCD + cd], dab, v[cd]);
        }
#pragma unroll
      for (int cd = 0; cd < NCD; ++cd) keep[cd * NT] += v[cd];
    }
    {  // K_ac += sum_bd g D_bd ; summed over the lanes of each ket half (they share c)
      double Dbd[NB * ND];
#pragma unroll
      for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int d = 0; d < ND; ++d) Dbd[b * ND + d] = D[(long)(b0 + b) * n + d0 + d];
      double v[NAT * NC];
#pragma unroll
      for (int a = 0; a < NAT; ++a)
#pragma unroll
        for (int c = 0; c < NC; ++c) {
          double sacc = 0.0;
#pragma unroll
          for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int d = 0; d < ND; ++d) sacc = fma(g[((a * NB + b) * NC + c) * ND + d], Dbd[b * ND + d], sacc);
          v[a * NC + c] = sacc;
        }
      warp_reduce_values<NAT * NC, true>(v, stage, x, [&](int vi, int half, double sum) { atomic_add(Km + (long)(a0 + vi / NC) * n + (half ? c0_hi : c0_lo) + vi % NC, sum); });
    }
    {  // K_ad += sum_bc g D_bc ; kept per lane over the rows (they share a).  D_bc is the same for all lanes
      double v[NAT * ND];
#pragma unroll
      for (int e = 0; e < NAT * ND; ++e) v[e] = 0.0;
#pragma unroll
      for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int c = 0; c < NC; ++c) {
          const double dbc = D[(long)(b0 + b) * n + c0 + c];
#pragma unroll
          for (int a = 0; a < NAT; ++a)
#pragma unroll
            for (int d = 0; d < ND; ++d) v[a * ND + d] = fma(g[((a * NB + b) * NC + c) * ND + d], dbc, v[a * ND + d]);
        }
#pragma unroll
      for (int e = 0; e < NAT * ND; ++e) keep[(NCD + e) * NT] += v[e];
    }
    {  // K_bc += sum_ad g D_ad ; summed over the lanes of each ket half
      double Dad[NAT * ND];
#pragma unroll
      for (int a = 0; a < NAT; ++a)
#pragma unroll
        for (int d = 0; d < ND; ++d) Dad[a * ND + d] = hold[(NCD + a * ND + d) * NT];
      double v[NB * NC];
#pragma unroll
      for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int c = 0; c < NC; ++c) {
          double sacc = 0.0;
#pragma unroll
          for (int a = 0; a < NAT; ++a)
#pragma unroll
            for (int d = 0; d < ND; ++d) sacc = fma(g[((a * NB + b) * NC + c) * ND + d], Dad[a * ND + d], sacc);
          v[b * NC + c] = sacc;
        }
      warp_reduce_values<NB * NC, true>(v, stage, x, [&](int vi, int half, double sum) { atomic_add(Km + (long)(b0 + vi / NC) * n + (half ? c0_hi : c0_lo) + vi % NC, sum); });
    }
    if (active) {  // K_bd += sum_ac g D_ac ; private to the quartet
      double v[NB * ND];
#pragma unroll
      for (int e = 0; e < NB * ND; ++e) v[e] = 0.0;
#pragma unroll
      for (int a = 0; a < NAT; ++a)
#pragma unroll
        for (int c = 0; c < NC; ++c) {
          const double dac = D[(long)(a0 + a) * n + c0 + c];
#pragma unroll
          for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int d = 0; d < ND; ++d) v[b * ND + d] = fma(g[((a * NB + b) * NC + c) * ND + d], dac, v[b * ND + d]);
        }
#pragma unroll
      for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int d = 0; d < ND; ++d) atomic_add(Km + (long)(b0 + b) * n + d0 + d, v[b * ND + d]);
    }
  }

  // ---- block end: J_cd summed over all warps, K_ad over the warps of the same team member; one atomic per element ----
  __syncthreads();
  const double* kall = smem + Tr::RT + Tr::NW * Tr::STAGE;
  for (int o = tid; o < NCD * 32; o += NT) {
    const int e = o >> 5, lane = o & 31;
    double sum = 0.0;
#pragma unroll
    for (int ww = 0; ww < Tr::NW; ++ww) sum += kall[e * NT + ww * 32 + lane];
    if (sum != 0.0) {
      const int2 cdl = kp.ao[j_first + lane];
      atomic_add(Jm + (long)(cdl.x + e / ND) * n + cdl.y + e % ND, sum);
    }
  }
  {
    const int a_first = bp.ao[i_first].x;
    for (int o = tid; o < NAT * ND * TQ * 32; o += NT) {
      const int lane = o & 31, rest = o >> 5, tt = rest % TQ, e = rest / TQ;   // e = a * ND + d
      double sum = 0.0;
#pragma unroll
      for (int gg = 0; gg < BI; ++gg) sum += kall[(NCD + e) * NT + (gg * TQ + tt) * 32 + lane];
      if (sum != 0.0) {
        const int2 cdl = kp.ao[j_first + lane];
        atomic_add(Km + (long)(a_first + tt * NAT + e / ND) * n + cdl.y + e % ND, sum);
      }
    }
  }
}

template <int LA, int LB, int LC, int LD, int TQ, int BI>
cudaError_t launch_tile_jk(const Work& w, int nblocks_dense, cudaStream_t s) {
  using Tr = TileTraits<LA, LB, LC, LD, TQ, BI>;
  const int grid = (nblocks_dense + w.nshard - 1) / w.nshard;
  if (grid <= 0) return cudaSuccess;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(tile_jk_kernel<LA, LB, LC, LD, TQ, BI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tr::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  tile_jk_kernel<LA, LB, LC, LD, TQ, BI><<<grid, dim3(32, BI * TQ), Tr::SMEM, s>>>(w);
  return cudaGetLastError();
}

}  // namespace eri
