// reg_kernel.cuh -- register family of J/K kernels (family R).
// One thread per shell quartet, angular momenta are template parameters, every loop over Cartesian components and
// recurrence indices is unrolled at compile time so that the 2-D integrals of one root and the contracted Cartesian
// block (ab|cd) live in registers (the paper's design rule 1, PAPER.md:59, PAPER.md:123 -- kept: it still holds on
// sm_100a).  What differs from the paper's Algorithm 2:
//   * contract, then digest ONCE per quartet into six small per-thread blocks (not six atomics per element);
//   * J_ab is summed over the 32 ket pairs of the warp with shuffles, J_cd over the bra rows of the block in shared
//     memory, so FP64 atomics are issued once per tile edge; only the four K blocks go out per quartet;
//   * digestion is in the Cartesian AO basis (D, J, K are transformed at matrix level once per call, transform.cu).
// Restricted to lb <= 1 and ld <= 1: the horizontal transfer then moves at most one quantum and needs no choice of
// build centre (the loss is (alpha_b/alpha_a)^lb relative, <= 1e-13 for any input).
#pragma once
#include "eri_dev.cuh"
#include "launch.h"

namespace eri {

constexpr int REG_BJ = 32, REG_BI = 4;   // block = 32 ket pairs (lanes) x 4 bra pairs (warps)

// 2-D integrals of one axis and one root, G[((i*(LB+1)+j)*(LC+1)+k)*(LD+1)+l] (reading R5).
template <int LA, int LB, int LC, int LD>
__device__ __forceinline__ void fill_2d_reg(double* __restrict__ G, double init, double c00, double c00p, double b10,
                                            double b01, double b00, double ab, double cd) {
  constexpr int NM = LA + LB, MM = LC + LD;
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
  // bra transfer (at most one quantum): B[i][j][m]
  double B[LA + 1][LB + 1][MM + 1];
#pragma unroll
  for (int m = 0; m <= MM; ++m) {
#pragma unroll
    for (int i = 0; i <= LA; ++i) {
      B[i][0][m] = T[i][m];
      if (LB == 1) B[i][LB][m] = fma(ab, T[i][m], T[i + 1][m]);
    }
  }
#pragma unroll
  for (int i = 0; i <= LA; ++i)
#pragma unroll
    for (int j = 0; j <= LB; ++j)
#pragma unroll
      for (int k = 0; k <= LC; ++k) {
        G[((i * (LB + 1) + j) * (LC + 1) + k) * (LD + 1)] = B[i][j][k];
        if (LD == 1) G[((i * (LB + 1) + j) * (LC + 1) + k) * (LD + 1) + 1] = fma(cd, B[i][j][k], B[i][j][k + 1]);
      }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(REG_BJ * REG_BI) reg_jk_kernel(Work w) {
  static_assert(LB <= 1 && LD <= 1, "register family: lb, ld <= 1");
  constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
  constexpr int NAB = NA * NB, NCD = NC * ND, NE = NAB * NCD;
  constexpr int N = nroots_of(LA + LB + LC + LD);
  constexpr int G2 = (LA + 1) * (LB + 1) * (LC + 1) * (LD + 1);
  constexpr int SB = (LC + 1) * (LD + 1), SA = (LB + 1) * SB, SC = LD + 1;
  __shared__ double red[NCD * REG_BI * REG_BJ];
  extern __shared__ __align__(16) double rtab[];   // Rys table of the class (eri_dev.cuh "Shared-memory copy"), dynamic shared memory
  rys_stage_table<N>(rtab, w.rys, threadIdx.y * REG_BJ + threadIdx.x, REG_BJ * REG_BI);
  __syncthreads();

  const PairSet& bp = w.bra; const PairSet& kp = w.ket;
  const int blk = blockIdx.x * w.nshard + w.shard;
  const bool list = w.list != nullptr;
  int i = 0, j = 0; double f = 0.0; bool active = false;
  if (list) {
    const long t = (long)blk * (REG_BJ * REG_BI) + threadIdx.y * REG_BJ + threadIdx.x;
    if (t < w.nlist) { i = w.list[t].x; j = w.list[t].y; f = 1.0; active = true; }
  } else if (blk < w.row_off[w.nrows]) {
    const int r = find_row(w.row_off, w.nrows, blk);
    i = r * REG_BI + threadIdx.y;
    j = (blk - w.row_off[r]) * REG_BJ + threadIdx.x;
    if (i < bp.npair && j < w.ket_count[i]) {
      active = true;
      f = bp.geom[6 * bp.stride + i] * kp.geom[6 * kp.stride + j];
      if (w.same && i == j) f *= 0.5;
    }
    if (i >= bp.npair) i = bp.npair - 1;   // keep the loads of idle threads in range
    if (j >= kp.npair) j = kp.npair - 1;
  }

  double g[NE];
#pragma unroll
  for (int e = 0; e < NE; ++e) g[e] = 0.0;

  if (active) {
    double A[3], AB[3], C[3], CD[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) {
      A[x] = bp.geom[x * bp.stride + i]; AB[x] = bp.geom[(3 + x) * bp.stride + i];
      C[x] = kp.geom[x * kp.stride + j]; CD[x] = kp.geom[(3 + x) * kp.stride + j];
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
        const double x = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
        const double pref = Kab * Kcd * sqrt(rpq);
        const double hq = 0.5 / q;
        double u[N], wt[N];
        rys_roots_smem<N>(x, rtab, w.rys, u, wt);
#pragma unroll
        for (int r = 0; r < N; ++r) {
          const double t2 = u[r] * rpq;          // u / (p+q)
          const double b00 = 0.5 * t2;
          const double b10 = hp - q * t2 * hp;   // (1 - q u/(p+q)) / 2p
          const double b01 = hq - p * t2 * hq;
          double gx[G2], gy[G2], gz[G2];
          fill_2d_reg<LA, LB, LC, LD>(gx, 1.0, (P[0] - A[0]) - q * t2 * PQ[0], (Q[0] - C[0]) + p * t2 * PQ[0], b10, b01, b00, AB[0], CD[0]);
          fill_2d_reg<LA, LB, LC, LD>(gy, 1.0, (P[1] - A[1]) - q * t2 * PQ[1], (Q[1] - C[1]) + p * t2 * PQ[1], b10, b01, b00, AB[1], CD[1]);
          fill_2d_reg<LA, LB, LC, LD>(gz, pref * wt[r], (P[2] - A[2]) - q * t2 * PQ[2], (Q[2] - C[2]) + p * t2 * PQ[2], b10, b01, b00, AB[2], CD[2]);
          int e = 0;
#pragma unroll
          for (int ax = LA; ax >= 0; --ax)
#pragma unroll
          for (int ay = LA - ax; ay >= 0; --ay)
#pragma unroll
          for (int bx = LB; bx >= 0; --bx)
#pragma unroll
          for (int by = LB - bx; by >= 0; --by)
#pragma unroll
          for (int cx = LC; cx >= 0; --cx)
#pragma unroll
          for (int cy = LC - cx; cy >= 0; --cy)
#pragma unroll
          for (int dx = LD; dx >= 0; --dx)
#pragma unroll
          for (int dy = LD - dx; dy >= 0; --dy) {
            const int az = LA - ax - ay, bz = LB - bx - by, cz = LC - cx - cy, dz = LD - dx - dy;
            g[e] = fma(gx[ax * SA + bx * SB + cx * SC + dx] * gy[ay * SA + by * SB + cy * SC + dy], gz[az * SA + bz * SB + cz * SC + dz], g[e]);
            ++e;
          }
        }
      }
    }
#pragma unroll
    for (int e = 0; e < NE; ++e) g[e] *= f;
  }

  // ---- digestion: the six updates of Alg. 2 lines 8-13, one small block at a time -----------
  const int n = w.nao;
  const int a0 = bp.ao[i].x, b0 = bp.ao[i].y, c0 = kp.ao[j].x, d0 = kp.ao[j].y;
  const double* __restrict__ D = w.D;
  {  // J_ab += sum_cd g D_cd : lanes of a warp share the bra pair in dense mode -> shuffle sum, one atomic per warp
    double Dcd[NCD];
#pragma unroll
    for (int c = 0; c < NC; ++c)
#pragma unroll
      for (int d = 0; d < ND; ++d) Dcd[c * ND + d] = D[(long)(c0 + c) * n + d0 + d];
#pragma unroll
    for (int ab = 0; ab < NAB; ++ab) {
      double s = 0.0;
#pragma unroll
      for (int cd = 0; cd < NCD; ++cd) s = fma(g[ab * NCD + cd], Dcd[cd], s);
      if (list) { if (active) atomic_add(w.J + (long)(a0 + ab / NB) * n + b0 + ab % NB, s); }
      else {
        s = warp_sum(s);
        if (threadIdx.x == 0) atomic_add(w.J + (long)(a0 + ab / NB) * n + b0 + ab % NB, s);
      }
    }
  }
  {  // J_cd += sum_ab g D_ab : the bra rows of the block share the ket pair in dense mode -> shared-memory sum
    double Dab[NAB];
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
      for (int b = 0; b < NB; ++b) Dab[a * NB + b] = D[(long)(a0 + a) * n + b0 + b];
#pragma unroll
    for (int cd = 0; cd < NCD; ++cd) {
      double s = 0.0;
#pragma unroll
      for (int ab = 0; ab < NAB; ++ab) s = fma(g[ab * NCD + cd], Dab[ab], s);
      if (list) { if (active) atomic_add(w.J + (long)(c0 + cd / ND) * n + d0 + cd % ND, s); }
      else red[(cd * REG_BI + threadIdx.y) * REG_BJ + threadIdx.x] = s;
    }
    if (!list) {
      __syncthreads();
      // thread (ty, tx) sums the values cd = ty, ty + BI, ... of ket lane tx
      for (int cd = threadIdx.y; cd < NCD; cd += REG_BI) {
        double s = 0.0;
#pragma unroll
        for (int y = 0; y < REG_BI; ++y) s += red[(cd * REG_BI + y) * REG_BJ + threadIdx.x];
        if (s != 0.0) atomic_add(w.J + (long)(c0 + cd / ND) * n + d0 + cd % ND, s);
      }
    }
  }
  if (!active) return;
  {  // K_ac += sum_bd g D_bd
    double Dbd[NB * ND];
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
      for (int d = 0; d < ND; ++d) Dbd[b * ND + d] = D[(long)(b0 + b) * n + d0 + d];
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
      for (int c = 0; c < NC; ++c) {
        double s = 0.0;
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
          for (int d = 0; d < ND; ++d) s = fma(g[((a * NB + b) * NC + c) * ND + d], Dbd[b * ND + d], s);
        atomic_add(w.K + (long)(a0 + a) * n + c0 + c, s);
      }
  }
  {  // K_ad += sum_bc g D_bc
    double Dbc[NB * NC];
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
      for (int c = 0; c < NC; ++c) Dbc[b * NC + c] = D[(long)(b0 + b) * n + c0 + c];
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
      for (int d = 0; d < ND; ++d) {
        double s = 0.0;
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
          for (int c = 0; c < NC; ++c) s = fma(g[((a * NB + b) * NC + c) * ND + d], Dbc[b * NC + c], s);
        atomic_add(w.K + (long)(a0 + a) * n + d0 + d, s);
      }
  }
  {  // K_bc += sum_ad g D_ad
    double Dad[NA * ND];
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
      for (int d = 0; d < ND; ++d) Dad[a * ND + d] = D[(long)(a0 + a) * n + d0 + d];
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
      for (int c = 0; c < NC; ++c) {
        double s = 0.0;
#pragma unroll
        for (int a = 0; a < NA; ++a)
#pragma unroll
          for (int d = 0; d < ND; ++d) s = fma(g[((a * NB + b) * NC + c) * ND + d], Dad[a * ND + d], s);
        atomic_add(w.K + (long)(b0 + b) * n + c0 + c, s);
      }
  }
  {  // K_bd += sum_ac g D_ac
    double Dac[NA * NC];
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
      for (int c = 0; c < NC; ++c) Dac[a * NC + c] = D[(long)(a0 + a) * n + c0 + c];
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
      for (int d = 0; d < ND; ++d) {
        double s = 0.0;
#pragma unroll
        for (int a = 0; a < NA; ++a)
#pragma unroll
          for (int c = 0; c < NC; ++c) s = fma(g[((a * NB + b) * NC + c) * ND + d], Dac[a * NC + c], s);
        atomic_add(w.K + (long)(b0 + b) * n + d0 + d, s);
      }
  }
}

template <int LA, int LB, int LC, int LD>
cudaError_t launch_reg_jk(const Work& w, int nblocks_dense, cudaStream_t s) {
  const int total = w.list ? (w.nlist + REG_BJ * REG_BI - 1) / (REG_BJ * REG_BI) : nblocks_dense;
  const int grid = (total + w.nshard - 1) / w.nshard;
  if (grid <= 0) return cudaSuccess;
  constexpr size_t rt_bytes = sizeof(double) * rys2_size(nroots_of(LA + LB + LC + LD));   // < 48 KB with the static part: no attribute needed
  reg_jk_kernel<LA, LB, LC, LD><<<grid, dim3(REG_BJ, REG_BI), rt_bytes, s>>>(w);
  return cudaGetLastError();
}

}  // namespace eri
