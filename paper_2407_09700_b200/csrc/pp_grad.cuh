// pp_grad.cuh -- primitive-parallel J/K gradient kernel (Algorithm 4; Eq. 11-15) for the
// deeply contracted units of the low-l classes: few shell quartets, each a sum over many primitive quartets (the K = 8 core s
// shells of the cfg3/cfg4 basis give 64 primitive ket pairs, up to 4096 primitive quartets per quartet).
// The tile gradient kernel (one THREAD per quartet) finds too few quartets in such units to fill its lanes, and the cooperative
// gradient kernel (one WARP per quartet, lane = (root, axis) in phase 1, lane = element in phase 2) keeps 3-6 of 32 lanes busy
// for 3-9 Cartesian elements: profiles/r02_cfg4.md, (ps|ss) K = 1,8,8,8 at 2.8 % of the FP64 peak.  Here a warp still owns a
// quartet (or several, see below), but its LANES OWN PRIMITIVE QUARTETS: lane l evaluates primitive quartets l, l + 32, ... completely in registers
// (roots from the shared-memory Rys table, 2-D integrals of one differentiated axis at a time, exactly the thread body of the
// tile gradient kernel), the density products pj = D_ab D_cd, pk = D_ac D_bd + D_ad D_bc are the same for all lanes and sit
// in a small shared-memory array per warp (broadcast loads), and the 18 scalars of the lanes are summed once per quartet.
// Task shape, screening and the treatment of centres C and D are those of the cooperative gradient kernel (coop_grad.cuh).
// The horizontal transfer is built on the first centre of each pair: the host selects this kernel only where that is safe.
#pragma once
#include "tile_grad.cuh"

namespace eri {

constexpr int PGRAD_WARPS = 4;   // ket pairs per block

constexpr int PGRAD_MAX_SUB = 10;   // quartets a warp evaluates side by side (3 primitive quartets each: 30 lanes)

template <int LA, int LB, int LC, int LD>
struct PPGradTraits {
  static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD), NE = NA * NB * NC * ND;
  static constexpr int N = nroots_of(LA + LB + LC + LD + 1);
  static constexpr int RT = rys2_size(N);
  static constexpr int PERWARP = 32 * 33 + 2 * NE * PGRAD_MAX_SUB;   // reduction staging + pj, pk of the warp's quartets
  static constexpr size_t SMEM = sizeof(double) * (RT + PGRAD_WARPS * PERWARP);
};

// Quartets with fewer than 32 primitive quartets share a warp: with npq primitive quartets per quartet the warp takes
// SUB = 32 / npq bra pairs of its task at a time and lane g * npq + t owns primitive quartet t of the g-th of them (npq = 8:
// four quartets, all lanes busy; npq = 3: ten quartets on 30 lanes).  Every group has its own density products; the 18 scalars
// are summed per group for centres A and B (they differ from bra pair to bra pair) and over the whole warp for C and D.
template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(32 * PGRAD_WARPS) pp_grad_kernel(Work w) {
  using Tr = PPGradTraits<LA, LB, LC, LD>;
  constexpr int NA = Tr::NA, NB = Tr::NB, NC = Tr::NC, ND = Tr::ND, NE = Tr::NE, N = Tr::N;
  extern __shared__ __align__(16) double smem[];
  const int lane = threadIdx.x, wy = threadIdx.y;
  const PairSet& bp = w.bra; const PairSet& kp = w.ket;
  const int blk = blockIdx.x * w.nshard + w.shard;
  if (blk >= w.row_off[w.nrows]) return;                     // block-uniform
  const double* rtab = smem;
  rys_stage_table<N>(smem, w.rys, wy * 32 + lane, 32 * PGRAD_WARPS);
  __syncthreads();
  double* stage = smem + Tr::RT + wy * Tr::PERWARP;
  double* pjk_all = stage + 32 * 33;                         // group g: pj[e] at g 2 NE + e, pk[e] at g 2 NE + NE + e

  const int r = find_row_warp(w.row_off, w.nrows, blk, lane);
  const int j = (blk - w.row_off[r]) * PGRAD_WARPS + wy;
  const int i_begin = r * w.grad_ch, i_end = min(i_begin + w.grad_ch, bp.npair);
  if (j >= kp.npair) return;                                 // whole warp, after the only block barrier
  const int n = w.nao;
  const double* __restrict__ D = w.D;
  double C[3], CD[3];
#pragma unroll
  for (int x = 0; x < 3; ++x) { C[x] = kp.geom[x * kp.stride + j]; CD[x] = kp.geom[(3 + x) * kp.stride + j]; }
  const double wket = kp.geom[6 * kp.stride + j];
  const int c0 = kp.ao[j].x, d0 = kp.ao[j].y;
  const int nppb = bp.npp, nppk = kp.npp, npq = nppb * nppk;
  const int GL = npq < 32 ? npq : 32;                                    // lanes of a group
  const int SUB = min(32 / GL, PGRAD_MAX_SUB);                           // quartets side by side
  const int g = lane / GL, gl = lane - g * GL;                           // this lane's group and place in it
  const bool in_group = g < SUB;
  double* pjk = pjk_all + (in_group ? g : 0) * 2 * NE;
  double keepC = 0.0, keepD = 0.0;   // lane v < 18: centre-C sum of value v and its share of centre D, over the task

  // the bra pairs of the task that have this ket pair in their kept prefix (at most 16 of them: CGRAD_CH)
  const int cand = i_begin + lane;
  const unsigned valid = __ballot_sync(0xffffffffu, cand < i_end && j < w.ket_count[cand]);
  const int nvalid = __popc(valid);

  for (int first = 0; first < nvalid; first += SUB) {
    const int mine = first + g;                              // which valid bra pair this lane's group takes
    const bool work = in_group && mine < nvalid;
    const int i = work ? i_begin + (int)__fns(valid, 0, mine + 1) : i_begin;
    double acc[18];   // [J: A xyz, B xyz, C xyz | K: same]
#pragma unroll
    for (int e = 0; e < 18; ++e) acc[e] = 0.0;
    __syncwarp();
    if (work) {   // density products of the group's quartet, once, for its lanes
      const int a0 = bp.ao[i].x, b0 = bp.ao[i].y;
      for (int e = gl; e < NE; e += GL) {
        const int d = e % ND, t1 = e / ND, c = t1 % NC, t2 = t1 / NC, b = t2 % NB, a = t2 / NB;
        const long ra = (long)(a0 + a) * n, rb = (long)(b0 + b) * n;
        pjk[e] = D[ra + b0 + b] * D[(long)(c0 + c) * n + d0 + d];
        pjk[NE + e] = fma(D[ra + c0 + c], D[rb + d0 + d], D[ra + d0 + d] * D[rb + c0 + c]);
      }
    }
    __syncwarp();
    if (work) {
      double f = bp.geom[6 * bp.stride + i] * wket;
      if (w.same && i == j) f *= 0.5;
      double A[3], AB[3];
#pragma unroll
      for (int x = 0; x < 3; ++x) { A[x] = bp.geom[x * bp.stride + i]; AB[x] = bp.geom[(3 + x) * bp.stride + i]; }
#pragma unroll 1
      for (int pq = gl; pq < npq; pq += GL) {
        const int kb = pq / nppk, kk = pq - kb * nppk;
        const double p = bp.prim[(kb * 5 + 0) * bp.stride + i];
        const double P[3] = {bp.prim[(kb * 5 + 1) * bp.stride + i], bp.prim[(kb * 5 + 2) * bp.stride + i], bp.prim[(kb * 5 + 3) * bp.stride + i]};
        const double Kab = bp.prim[(kb * 5 + 4) * bp.stride + i];
        const double ea2 = 2.0 * bp.aexp[(kb * 2 + 0) * bp.stride + i], eb2 = 2.0 * bp.aexp[(kb * 2 + 1) * bp.stride + i];
        const double q = kp.prim[(kk * 5 + 0) * kp.stride + j];
        const double Q[3] = {kp.prim[(kk * 5 + 1) * kp.stride + j], kp.prim[(kk * 5 + 2) * kp.stride + j], kp.prim[(kk * 5 + 3) * kp.stride + j]};
        const double Kcd = kp.prim[(kk * 5 + 4) * kp.stride + j];
        const double ec2 = 2.0 * kp.aexp[(kk * 2 + 0) * kp.stride + j];
        const double hp = 0.5 / p, hq = 0.5 / q;
        const double rpq = 1.0 / (p + q), rho = p * q * rpq;
        const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
        const double xx = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
        const double pref = f * Kab * Kcd * sqrt(rpq);
        double u[N], wt[N];
        rys_roots_smem<N>(xx, rtab, w.rys, u, wt);
#pragma unroll 1
        for (int rt = 0; rt < N; ++rt) {
          const double t2 = u[rt] * rpq;
          const double b00 = 0.5 * t2, b10 = hp - q * t2 * hp, b01 = hq - p * t2 * hq;
          const double c00[3] = {(P[0] - A[0]) - q * t2 * PQ[0], (P[1] - A[1]) - q * t2 * PQ[1], (P[2] - A[2]) - q * t2 * PQ[2]};
          const double c00p[3] = {(Q[0] - C[0]) + p * t2 * PQ[0], (Q[1] - C[1]) + p * t2 * PQ[1], (Q[2] - C[2]) + p * t2 * PQ[2]};
          const double init[3] = {1.0, 1.0, pref * wt[rt]};
          // one differentiated axis per trip of a loop that is NOT unrolled: inlined back to back, the three axis bodies share
          // their 2 NE loads of pj, pk as common subexpressions, the compiler keeps them in registers across the bodies and spills
          // (pp_grad_kernel<2,1,1,0>: 1.5 KB of spill stores per thread, 15.7 GB of DRAM traffic per cfg4 step, profiles/r02_cfg4.md)
#pragma unroll 1
          for (int axis = 0; axis < 3; ++axis) {
            double a6[6];
#pragma unroll
            for (int e = 0; e < 6; ++e) a6[e] = 0.0;
            switch (axis) {
              case 0:
                tile_grad_team_axis<LA, LB, LC, LD, 0, 1>(a6, c00, c00p, init, b10, b01, b00, AB, CD, ea2, eb2, ec2, pjk);
#pragma unroll
                for (int e = 0; e < 6; ++e) acc[(e / 3) * 9 + (e % 3) * 3 + 0] += a6[e];
                break;
              case 1:
                tile_grad_team_axis<LA, LB, LC, LD, 1, 1>(a6, c00, c00p, init, b10, b01, b00, AB, CD, ea2, eb2, ec2, pjk);
#pragma unroll
                for (int e = 0; e < 6; ++e) acc[(e / 3) * 9 + (e % 3) * 3 + 1] += a6[e];
                break;
              default:
                tile_grad_team_axis<LA, LB, LC, LD, 2, 1>(a6, c00, c00p, init, b10, b01, b00, AB, CD, ea2, eb2, ec2, pjk);
#pragma unroll
                for (int e = 0; e < 6; ++e) acc[(e / 3) * 9 + (e % 3) * 3 + 2] += a6[e];
                break;
            }
          }
        }
      }
    }
    // PJ = 4 f ..., PK = 2 f ... (f is in the prefactor).  The lanes stage their 18 scalars (value-row major); centres A and B
    // are summed per group and leave now, lane v < 18 adds the warp's total of value v to its C sum and its share of centre D
#pragma unroll
    for (int e = 0; e < 9; ++e) { acc[e] *= 4.0; acc[9 + e] *= 2.0; }
    if (SUB == 1) {   // one quartet per warp: the 18 sums over the lanes as in the cooperative gradient kernel
      const int2 at_ab = bp.atom[i_begin + (int)__fns(valid, 0, first + 1)];   // (lanes beyond the group hold no bra pair)
      warp_reduce_values<18, false>(acc, stage, lane, [&](int v, int, double sum) {
        const int jk = v / 9, ce = (v % 9) / 3, ax = v % 3;
        if (ce < 2) atomic_add((jk ? w.gK : w.gJ) + 3 * (ce == 0 ? at_ab.x : at_ab.y) + ax, sum);
        else keepC += sum;
        keepD -= sum;
      });
      continue;
    }
#pragma unroll
    for (int e = 0; e < 18; ++e) stage[e * 33 + lane] = acc[e];
    __syncwarp();
    const int ngrp = min(SUB, nvalid - first);
    for (int it = lane; it < 12 * ngrp; it += 32) {
      const int gg = it / 12, v12 = it - gg * 12;                 // v12 = jk * 6 + centre * 3 + axis, centre in {A, B}
      const int jk = v12 / 6, ce = (v12 % 6) / 3, ax = v12 % 3;
      const double* src = stage + (jk * 9 + ce * 3 + ax) * 33 + gg * GL;
      double sum = 0.0;
      for (int l = 0; l < GL; ++l) sum += src[l];
      const int2 at_ab = bp.atom[i_begin + (int)__fns(valid, 0, first + gg + 1)];
      if (sum != 0.0) atomic_add((jk ? w.gK : w.gJ) + 3 * (ce == 0 ? at_ab.x : at_ab.y) + ax, sum);
    }
    if (lane < 18) {
      const double* src = stage + lane * 33;
      double sum = 0.0;
      for (int l = 0; l < ngrp * GL; ++l) sum += src[l];
      if ((lane % 9) / 3 == 2) keepC += sum;
      keepD -= sum;
    }
  }
  if (lane < 18) {
    const int jk = lane / 9, ax = lane % 3;
    const int2 at_cd = kp.atom[j];
    double* gout = jk ? w.gK : w.gJ;
    if (keepC != 0.0) atomic_add(gout + 3 * at_cd.x + ax, keepC);
    if (keepD != 0.0) atomic_add(gout + 3 * at_cd.y + ax, keepD);
  }
}

template <int LA, int LB, int LC, int LD>
cudaError_t launch_pp_grad(const Work& w, int nblocks_dense, cudaStream_t s) {
  using Tr = PPGradTraits<LA, LB, LC, LD>;
  static_assert(Tr::SMEM <= 227 * 1024, "primitive-parallel gradient kernel: shared memory");
  const int grid = (nblocks_dense + w.nshard - 1) / w.nshard;
  if (grid <= 0) return cudaSuccess;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(pp_grad_kernel<LA, LB, LC, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tr::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  pp_grad_kernel<LA, LB, LC, LD><<<grid, dim3(32, PGRAD_WARPS), Tr::SMEM, s>>>(w);
  return cudaGetLastError();
}

}  // namespace eri
