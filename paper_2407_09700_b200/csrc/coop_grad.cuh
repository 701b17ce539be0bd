// coop_grad.cuh -- cooperative family, J/K gradient kernel (Algorithm 4; Eq. 11-15)
// for the classes whose unrolled thread-per-quartet body (tile_grad.cuh) does not fit the register file.
// One WARP per shell quartet, as in coop_kernel.cuh:
//   phase 1  lane (root r, axis x) builds the 2-D integrals with the indices of centres A, B, C raised by one
//            (centre D follows from translational invariance) on the numerically safe centres and stores
//            them to the warp's shared-memory slab S[axis][root][i][j][k][l];
//   phase 2  lane `ab` owns a Cartesian bra component pair; for every ket component pair and root it forms
//            F[I] = 2 alpha I(+1) - n I(-1) (Eq. 11) on the three centres and three axes and adds
//            dI/dR . (PJ, PK) (reading R10/R11) into 18 per-lane scalars -- no per-element accumulator;
//   phase 3  the 18 scalars are summed over the lanes through the (dead) slab: centres A and B leave per quartet,
//            centres C and D are kept over the bra pairs of the warp's task and leave once per task.
// A task is one ket pair and a run of CH consecutive bra pairs of the Schwarz-sorted tile row (dense mode).
#pragma once
#include "coop_kernel.cuh"
#include "tile_kernel.cuh"   // warp_reduce_values

namespace eri {

constexpr int CGRAD_CH = 16;      // bra pairs per task (the host shortens the run, Work::grad_ch, for units of few heavy quartets)

// WARPS = ket pairs per block (gen_class_lists.py sizes it for 200 KB of shared memory).  EM = element mode of phase 2: the
// Cartesian elements (a,b,c,d) are dealt over the 32 lanes one by one (run-time component indices, density blocks staged in
// shared memory) instead of one bra component pair per lane -- for the classes whose nc(la) nc(lb) fills the lanes badly
// ((dp|, (dd|, (fs| ...: 18, 36, 10 pairs).  There is no per-element accumulator, so any distribution of the elements works.
template <int LA, int LB, int LC, int LD, int WARPS, int EM>
struct CoopGradTraits {
  static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
  static constexpr int NAB = NA * NB, NCD = NC * ND;
  static constexpr int PASSES = (NAB + 31) / 32;
  // ab-mode with a tail: when the last pass would hold at most 8 bra component pairs ((dd|: 36 = 32 + 4, (ff|: 100 = 96 + 4),
  // those pairs' elements are dealt over all lanes one by one (as in element mode) after the full passes
  static constexpr int REM = NAB % 32;
  static constexpr bool TAIL = EM == 0 && NAB > 32 && REM > 0 && REM <= 8;
  static constexpr int PASSES_AB = TAIL ? NAB / 32 : PASSES;
  static constexpr int N = nroots_of(LA + LB + LC + LD + 1);
  static constexpr int SCD = ((LC + 2) * (LD + 1)) | 1, G2 = ((LA + 2) * (LB + 2) * SCD) | 1;   // raised on A, B, C; odd strides: no bank conflicts
  static constexpr int SLAB2D = 3 * N * G2;
  static constexpr int BASE = SLAB2D > 32 * 33 ? SLAB2D : 32 * 33;
  static constexpr int NDQ = EM ? NAB + NA * NC + NA * ND + NB * NC + NB * ND : 0;   // D_ab, D_ac, D_ad, D_bc, D_bd of the quartet (element mode)
  // paired phase 1 as in coop_kernel.cuh: the two half-warps build the raised 2-D integrals of two consecutive primitive quartets
  // of the task, each into its own slab -- where the second slab does not cost a resident block (MINB3: the classes that hold
  // three blocks per SM by registers, the others hold two)
  static constexpr bool MINB3 = EM == 0 && WARPS == 4 && LD == 0 && LC >= 1 && LC <= 2 && NAB >= 18;   // three blocks per SM where measured faster (cfg4)
  static constexpr bool PAIR = 3 * N <= 16 && sizeof(double) * (BASE + SLAB2D + NDQ + NCD) * WARPS <= (MINB3 ? 75 : 113) * 1024;
  // dual phase 2 (paired kernels of the classes with 18 bra component pairs, (dp|): a pass of phase 2 kept 18 of 32 lanes busy.
  // Both slabs of a pair are consumed at once instead: half-warp h takes bra component pairs 0..15 of item h, and the two
  // remaining pairs of each item are dealt over the 16 lanes of its half element by element.
  // The classes with 9 to 16 bra component pairs run the same way (no remaining pairs): two items in ab-mode on 2 NAB lanes load a
  // sixth of what element mode loads from shared memory per element (gen_class_lists.py gives them EM = 0 where PAIR holds).
  static constexpr bool DUAL = PAIR && EM == 0 && NAB >= 9 && NAB <= 20;
  static constexpr int SLAB = BASE + (PAIR ? SLAB2D : 0) + NDQ + NCD;               // + second slab + staged density blocks
  static constexpr size_t SMEM = sizeof(double) * SLAB * WARPS;
  static_assert(SMEM <= 227 * 1024, "slab does not fit");
  static_assert(3 * N <= 32, "one lane per (root, axis)");
};

template <int LA, int LB, int LC, int LD, int WARPS, int EM>
__global__ void __launch_bounds__(32 * WARPS, (CoopGradTraits<LA, LB, LC, LD, WARPS, EM>::MINB3 ? 3 : 0)) coop_grad_kernel(Work w) {
  using Tr = CoopGradTraits<LA, LB, LC, LD, WARPS, EM>;
  constexpr int NA = Tr::NA, NB = Tr::NB, NC = Tr::NC, ND = Tr::ND, NAB = Tr::NAB, NCD = Tr::NCD, PASSES = Tr::PASSES;
  constexpr int N = Tr::N, SCD = Tr::SCD, G2 = Tr::G2;
  constexpr int SL = 1, SK = LD + 1, SJ = SCD, SI = (LB + 2) * SCD;   // strides of (i, j, k, l) in the slab
  extern __shared__ double smem[];
  const int lane = threadIdx.x, wy = threadIdx.y;
  double* S = smem + (size_t)wy * Tr::SLAB;
  double* sDcd = S + (Tr::SLAB - NCD);
  double* sDab = S + (Tr::SLAB - NCD - Tr::NDQ); double* sDac = sDab + NAB; double* sDad = sDac + NA * NC; double* sDbc = sDad + NA * ND; double* sDbd = sDbc + NB * NC;   // element mode

  const PairSet& bp = w.bra; const PairSet& kp = w.ket;
  const int blk = blockIdx.x * w.nshard + w.shard;
  if (blk >= w.row_off[w.nrows]) return;
  const int r = find_row_warp(w.row_off, w.nrows, blk, threadIdx.x);
  const int j = (blk - w.row_off[r]) * WARPS + wy;
  const int i_begin = r * w.grad_ch, i_end = min(i_begin + w.grad_ch, bp.npair);
  if (j >= kp.npair) return;
  const int n = w.nao;
  const double* __restrict__ D = w.D;

  // ---- per-task ket data ----
  double C[3], CD[3];
#pragma unroll
  for (int x = 0; x < 3; ++x) { C[x] = kp.geom[x * kp.stride + j]; CD[x] = kp.geom[(3 + x) * kp.stride + j]; }
  const double wket = kp.geom[6 * kp.stride + j];
  const int c0 = kp.ao[j].x, d0 = kp.ao[j].y;
  for (int cd = lane; cd < NCD; cd += 32) sDcd[cd] = D[(long)(c0 + cd / ND) * n + d0 + cd % ND];
  __syncwarp();

  const int my_root = lane / 3, my_axis = lane - 3 * my_root;
  const bool fill_lane = lane < 3 * N;
  double keepC = 0.0, keepD = 0.0;   // lane v < 18: centre-C sum of value v (if v is a C value) and its share of centre D, over the task

  double acc[18];   // [J: A xyz, B xyz, C xyz | K: same]
#pragma unroll
  for (int e = 0; e < 18; ++e) acc[e] = 0.0;

  // element mode: the five density blocks of the quartet (bra pair i) that involve a bra shell, staged in shared memory
  [[maybe_unused]] auto stage = [&](int i) {
    const int a0 = bp.ao[i].x, b0 = bp.ao[i].y;
    {
      __syncwarp();
      for (int e = lane; e < NAB; e += 32) sDab[e] = D[(long)(a0 + e / NB) * n + b0 + e % NB];
      for (int e = lane; e < NA * NC; e += 32) sDac[e] = D[(long)(a0 + e / NC) * n + c0 + e % NC];
      for (int e = lane; e < NA * ND; e += 32) sDad[e] = D[(long)(a0 + e / ND) * n + d0 + e % ND];
      for (int e = lane; e < NB * NC; e += 32) sDbc[e] = D[(long)(b0 + e / NC) * n + c0 + e % NC];
      for (int e = lane; e < NB * ND; e += 32) sDbd[e] = D[(long)(b0 + e / ND) * n + d0 + e % ND];
      __syncwarp();
    }

  };

  // ---- phase 2: the primitive quartet whose raised 2-D integrals are in the slab S2 adds to the 18 scalars ----------------
  // dual = true (Tr::DUAL only): S2, i and the exponents are those of the lane's half-warp (two items at once)
  auto phase2 = [&](const double* __restrict__ S2, int i, double ea2, double eb2, double ec2, bool dual) {
    [[maybe_unused]] const int a0 = bp.ao[i].x, b0 = bp.ao[i].y;
    if constexpr (EM != 0) {
#pragma unroll 1
      for (int e = lane; e < NAB * NCD; e += 32) {
        const int id = e % ND, t1 = e / ND, ic = t1 % NC, t2 = t1 / NC, ib = t2 % NB, ia = t2 / NB;
        int ax, ay, az, bx, by, bz, cx, cy, cz, dx, dy, dz;
        cart_powers(LA, ia, ax, ay, az); cart_powers(LB, ib, bx, by, bz); cart_powers(LC, ic, cx, cy, cz); cart_powers(LD, id, dx, dy, dz);
        const double pj = sDab[ia * NB + ib] * sDcd[ic * ND + id];
        const double pk = fma(sDac[ia * NC + ic], sDbd[ib * ND + id], sDad[ia * ND + id] * sDbc[ib * NC + ic]);
        const int ox = ax * SI + bx * SJ + cx * SK + dx, oy = ay * SI + by * SJ + cy * SK + dy + N * G2, oz = az * SI + bz * SJ + cz * SK + dz + 2 * N * G2;
        // lowered terms vanish with their integer factor; the slab has no index -1, so the offset is 0 there
        const int lax = ax > 0 ? -SI : 0, lay = ay > 0 ? -SI : 0, laz = az > 0 ? -SI : 0;
        const int lbx = bx > 0 ? -SJ : 0, lby = by > 0 ? -SJ : 0, lbz = bz > 0 ? -SJ : 0;
        const int lcx = cx > 0 ? -SK : 0, lcy = cy > 0 ? -SK : 0, lcz = cz > 0 ? -SK : 0;
        const double fax = ax, fay = ay, faz = az, fbx = bx, fby = by, fbz = bz, fcx = cx, fcy = cy, fcz = cz;
#pragma unroll 1
        for (int rt = 0; rt < N; ++rt) {
          const double* X = S2 + ox + rt * G2;
          const double* Y = S2 + oy + rt * G2;
          const double* Z = S2 + oz + rt * G2;
          const double vx = X[0], vy = Y[0], vz = Z[0];
          const double oyz = vy * vz, oxz = vx * vz, oxy = vx * vy;
          const double dAx = fma(ea2, X[SI], -fax * X[lax]), dAy = fma(ea2, Y[SI], -fay * Y[lay]), dAz = fma(ea2, Z[SI], -faz * Z[laz]);
          const double dBx = fma(eb2, X[SJ], -fbx * X[lbx]), dBy = fma(eb2, Y[SJ], -fby * Y[lby]), dBz = fma(eb2, Z[SJ], -fbz * Z[lbz]);
          const double dCx = fma(ec2, X[SK], -fcx * X[lcx]), dCy = fma(ec2, Y[SK], -fcy * Y[lcy]), dCz = fma(ec2, Z[SK], -fcz * Z[lcz]);
          const double jx = pj * oyz, jy = pj * oxz, jz = pj * oxy;
          const double kx = pk * oyz, ky = pk * oxz, kz = pk * oxy;
          acc[0] = fma(dAx, jx, acc[0]); acc[1] = fma(dAy, jy, acc[1]); acc[2] = fma(dAz, jz, acc[2]);
          acc[3] = fma(dBx, jx, acc[3]); acc[4] = fma(dBy, jy, acc[4]); acc[5] = fma(dBz, jz, acc[5]);
          acc[6] = fma(dCx, jx, acc[6]); acc[7] = fma(dCy, jy, acc[7]); acc[8] = fma(dCz, jz, acc[8]);
          acc[9] = fma(dAx, kx, acc[9]); acc[10] = fma(dAy, ky, acc[10]); acc[11] = fma(dAz, kz, acc[11]);
          acc[12] = fma(dBx, kx, acc[12]); acc[13] = fma(dBy, ky, acc[13]); acc[14] = fma(dBz, kz, acc[14]);
          acc[15] = fma(dCx, kx, acc[15]); acc[16] = fma(dCy, ky, acc[16]); acc[17] = fma(dCz, kz, acc[17]);
        }
      }
    } else {
#pragma unroll
    for (int ps = 0; ps < Tr::PASSES_AB; ++ps) {
      int ab = (Tr::DUAL && dual ? (lane & 15) : lane) + 32 * ps;
      const bool own = ab < NAB;
      if (!own) ab = NAB - 1;
      const int ia = ab / NB, ib = ab - ia * NB;
      int ax, ay, az, bx, by, bz;
      cart_powers(LA, ia, ax, ay, az); cart_powers(LB, ib, bx, by, bz);
      // D is symmetric: the blocks are read through their transposes (one row of D per load instruction instead of NA or NB rows,
      // coop_kernel.cuh phase 3)
      const int ca = a0 + ia, cb = b0 + ib;
      const double dab = own ? D[(long)cb * n + ca] : 0.0;
      double Dac[NC], Dbc[NC], Dad[ND], Dbd[ND];
#pragma unroll
      for (int c = 0; c < NC; ++c) { const long rc = (long)(c0 + c) * n; Dac[c] = own ? D[rc + ca] : 0.0; Dbc[c] = own ? D[rc + cb] : 0.0; }
#pragma unroll
      for (int d = 0; d < ND; ++d) { const long rd = (long)(d0 + d) * n; Dad[d] = D[rd + ca]; Dbd[d] = D[rd + cb]; }
      const int ox = (ax * SI + bx * SJ), oy = (ay * SI + by * SJ) + N * G2, oz = (az * SI + bz * SJ) + 2 * N * G2;
      const double fax = (double)ax, fay = (double)ay, faz = (double)az, fbx = (double)bx, fby = (double)by, fbz = (double)bz;
#pragma unroll 1
      for (int rt = 0; rt < N; ++rt) {
        const double* X = S2 + ox + rt * G2;
        const double* Y = S2 + oy + rt * G2;
        const double* Z = S2 + oz + rt * G2;
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
            const int ex = cx * SK + dx, ey = cy * SK + dy, ez = cz * SK + dz;
            const double vx = X[ex], vy = Y[ey], vz = Z[ez];
            const double oyz = vy * vz, oxz = vx * vz, oxy = vx * vy;
            // lowered terms vanish with their integer factor; the slab has no index -1, so guard the address
            const double dAx = fma(ea2, X[ex + SI], -fax * X[ax > 0 ? ex - SI : ex]);
            const double dAy = fma(ea2, Y[ey + SI], -fay * Y[ay > 0 ? ey - SI : ey]);
            const double dAz = fma(ea2, Z[ez + SI], -faz * Z[az > 0 ? ez - SI : ez]);
            const double dBx = fma(eb2, X[ex + SJ], -fbx * X[bx > 0 ? ex - SJ : ex]);
            const double dBy = fma(eb2, Y[ey + SJ], -fby * Y[by > 0 ? ey - SJ : ey]);
            const double dBz = fma(eb2, Z[ez + SJ], -fbz * Z[bz > 0 ? ez - SJ : ez]);
            const double dCx = cx > 0 ? fma(ec2, X[ex + SK], -cx * X[ex - SK]) : ec2 * X[ex + SK];
            const double dCy = cy > 0 ? fma(ec2, Y[ey + SK], -cy * Y[ey - SK]) : ec2 * Y[ey + SK];
            const double dCz = cz > 0 ? fma(ec2, Z[ez + SK], -cz * Z[ez - SK]) : ec2 * Z[ez + SK];
            const double pj = dab * sDcd[c * ND + d];
            const double pk = fma(Dac[c], Dbd[d], Dad[d] * Dbc[c]);
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
      }
    }
    if constexpr (Tr::TAIL || Tr::DUAL) {
      // the last NAB % 32 bra component pairs: their elements dealt over all lanes (there is no per-element accumulator, so any
      // distribution works) instead of one more pass that keeps NAB % 32 of 32 lanes busy -- (dd|: 4 of 32.  Dual phase 2: the
      // pairs from 16 on of the half-warp's item over the 16 lanes of the half
      const int tail_ab0 = Tr::DUAL ? 16 : 32 * Tr::PASSES_AB;
      const int tail_n = Tr::DUAL ? (dual ? (NAB - 16) * NCD : 0) : Tr::REM * NCD;
      const int tail_q = Tr::DUAL ? (lane & 15) : lane, tail_stride = Tr::DUAL ? 16 : 32;
#pragma unroll 1
      for (int e = tail_q; e < tail_n; e += tail_stride) {
        const int id = e % ND, t1 = e / ND, ic = t1 % NC, ab = tail_ab0 + t1 / NC, ib = ab % NB, ia = ab / NB;
        int ax, ay, az, bx, by, bz, cx, cy, cz, dx, dy, dz;
        cart_powers(LA, ia, ax, ay, az); cart_powers(LB, ib, bx, by, bz); cart_powers(LC, ic, cx, cy, cz); cart_powers(LD, id, dx, dy, dz);
        const long ra = (long)(a0 + ia) * n, rb = (long)(b0 + ib) * n;
        const double pj = D[ra + b0 + ib] * sDcd[ic * ND + id];
        const double pk = fma(D[ra + c0 + ic], D[rb + d0 + id], D[ra + d0 + id] * D[rb + c0 + ic]);
        const int ox = ax * SI + bx * SJ + cx * SK + dx, oy = ay * SI + by * SJ + cy * SK + dy + N * G2, oz = az * SI + bz * SJ + cz * SK + dz + 2 * N * G2;
        // lowered terms vanish with their integer factor; the slab has no index -1, so the offset is 0 there
        const int lax = ax > 0 ? -SI : 0, lay = ay > 0 ? -SI : 0, laz = az > 0 ? -SI : 0;
        const int lbx = bx > 0 ? -SJ : 0, lby = by > 0 ? -SJ : 0, lbz = bz > 0 ? -SJ : 0;
        const int lcx = cx > 0 ? -SK : 0, lcy = cy > 0 ? -SK : 0, lcz = cz > 0 ? -SK : 0;
        const double fax = ax, fay = ay, faz = az, fbx = bx, fby = by, fbz = bz, fcx = cx, fcy = cy, fcz = cz;
#pragma unroll 1
        for (int rt = 0; rt < N; ++rt) {
          const double* X = S2 + ox + rt * G2;
          const double* Y = S2 + oy + rt * G2;
          const double* Z = S2 + oz + rt * G2;
          const double vx = X[0], vy = Y[0], vz = Z[0];
          const double oyz = vy * vz, oxz = vx * vz, oxy = vx * vy;
          const double dAx = fma(ea2, X[SI], -fax * X[lax]), dAy = fma(ea2, Y[SI], -fay * Y[lay]), dAz = fma(ea2, Z[SI], -faz * Z[laz]);
          const double dBx = fma(eb2, X[SJ], -fbx * X[lbx]), dBy = fma(eb2, Y[SJ], -fby * Y[lby]), dBz = fma(eb2, Z[SJ], -fbz * Z[lbz]);
          const double dCx = fma(ec2, X[SK], -fcx * X[lcx]), dCy = fma(ec2, Y[SK], -fcy * Y[lcy]), dCz = fma(ec2, Z[SK], -fcz * Z[lcz]);
          const double jx = pj * oyz, jy = pj * oxz, jz = pj * oxy;
          const double kx = pk * oyz, ky = pk * oxz, kz = pk * oxy;
          acc[0] = fma(dAx, jx, acc[0]); acc[1] = fma(dAy, jy, acc[1]); acc[2] = fma(dAz, jz, acc[2]);
          acc[3] = fma(dBx, jx, acc[3]); acc[4] = fma(dBy, jy, acc[4]); acc[5] = fma(dBz, jz, acc[5]);
          acc[6] = fma(dCx, jx, acc[6]); acc[7] = fma(dCy, jy, acc[7]); acc[8] = fma(dCz, jz, acc[8]);
          acc[9] = fma(dAx, kx, acc[9]); acc[10] = fma(dAy, ky, acc[10]); acc[11] = fma(dAz, kz, acc[11]);
          acc[12] = fma(dBx, kx, acc[12]); acc[13] = fma(dBy, ky, acc[13]); acc[14] = fma(dBz, kz, acc[14]);
          acc[15] = fma(dCx, kx, acc[15]); acc[16] = fma(dCy, ky, acc[16]); acc[17] = fma(dCz, kz, acc[17]);
        }
      }
    }
    }
  };

  // ---- phase 3 of the finished quartet (bra pair i), then acc = 0 ---------------------------------------------------------
  auto phase3 = [&](int i) {
    // PJ = 4 f ..., PK = 2 f ... (f is in the prefactor); sum over the lanes through the dead slab (slab 0)
#pragma unroll
    for (int e = 0; e < 9; ++e) { acc[e] *= 4.0; acc[9 + e] *= 2.0; }
    const int2 at_ab = bp.atom[i];
    // lane v = jk*9 + centre*3 + axis receives the sum of value v: centres A, B leave now; the lane keeps its C sum and
    // its share of centre D = -(A + B + C) until the task ends
    warp_reduce_values<18, false>(acc, S, lane, [&](int v, int, double sum) {
      const int jk = v / 9, ce = (v % 9) / 3, ax = v % 3;
      if (ce < 2) atomic_add((jk ? w.gK : w.gJ) + 3 * (ce == 0 ? at_ab.x : at_ab.y) + ax, sum);
      else keepC += sum;
      keepD -= sum;
    });
    __syncwarp();
#pragma unroll
    for (int e = 0; e < 18; ++e) acc[e] = 0.0;
  };

  // dual phase 2 with one primitive quartet per quartet: lanes 0-15 hold the sums of bra pair ia, lanes 16-31 those of ib
  [[maybe_unused]] auto phase3_halves = [&](int ia, int ib) {
#pragma unroll
    for (int e = 0; e < 9; ++e) { acc[e] *= 4.0; acc[9 + e] *= 2.0; }
    const int2 at_a = bp.atom[ia], at_b = bp.atom[ib];
    warp_reduce_values<18, true>(acc, S, lane, [&](int v, int half, double sum) {
      const int jk = v / 9, ce = (v % 9) / 3, ax = v % 3;
      const int2 at_ab = half ? at_b : at_a;
      if (ce < 2) atomic_add((jk ? w.gK : w.gJ) + 3 * (ce == 0 ? at_ab.x : at_ab.y) + ax, sum);
      else keepC += sum;
      keepD -= sum;
    });
    __syncwarp();
#pragma unroll
    for (int e = 0; e < 18; ++e) acc[e] = 0.0;
  };

  if constexpr (!Tr::PAIR) {
  for (int i = i_begin; i < i_end; ++i) {
    if (j >= w.ket_count[i]) continue;     // warp-uniform
    double f = bp.geom[6 * bp.stride + i] * wket;
    if (w.same && i == j) f *= 0.5;
    double A[3], AB[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) { A[x] = bp.geom[x * bp.stride + i]; AB[x] = bp.geom[(3 + x) * bp.stride + i]; }
    if constexpr (EM != 0) stage(i);
    for (int kb = 0; kb < bp.npp; ++kb) {
      const double p = bp.prim[(kb * 5 + 0) * bp.stride + i];
      const double P[3] = {bp.prim[(kb * 5 + 1) * bp.stride + i], bp.prim[(kb * 5 + 2) * bp.stride + i], bp.prim[(kb * 5 + 3) * bp.stride + i]};
      const double Kab = bp.prim[(kb * 5 + 4) * bp.stride + i];
      const double ea2 = 2.0 * bp.aexp[(kb * 2 + 0) * bp.stride + i], eb2 = 2.0 * bp.aexp[(kb * 2 + 1) * bp.stride + i];
      bool swb;   // build on B when P is nearer to B (the raised index of B is always transferred)
      {
        double da = 0.0, db = 0.0;
#pragma unroll
        for (int x = 0; x < 3; ++x) { const double pa = P[x] - A[x], pb = pa + AB[x]; da += pa * pa; db += pb * pb; }
        swb = db < da;
      }
      for (int kk = 0; kk < kp.npp; ++kk) {
        const double q = kp.prim[(kk * 5 + 0) * kp.stride + j];
        const double Q[3] = {kp.prim[(kk * 5 + 1) * kp.stride + j], kp.prim[(kk * 5 + 2) * kp.stride + j], kp.prim[(kk * 5 + 3) * kp.stride + j]};
        const double Kcd = kp.prim[(kk * 5 + 4) * kp.stride + j];
        const double ec2 = 2.0 * kp.aexp[(kk * 2 + 0) * kp.stride + j];
        bool swk = false;
        if (LD > 0) {
          double dc = 0.0, dd = 0.0;
#pragma unroll
          for (int x = 0; x < 3; ++x) { const double qc = Q[x] - C[x], qd = qc + CD[x]; dc += qc * qc; dd += qd * qd; }
          swk = dd < dc;
        }
        const double rpq = 1.0 / (p + q), rho = p * q * rpq;
        const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
        const double xx = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
        // ---- phase 1 ----
        __syncwarp();
        if (fill_lane) {
          double u, wt;
          rys_root_one<N>(xx, w.rys, my_root, u, wt);
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
          const double init = ax == 2 ? f * Kab * Kcd * sqrt(rpq) * wt : 1.0;
          double* dst = S + (ax * N + my_root) * G2;
          if (!swb) {
            if (!swk) fill_2d_smem<LA + 1, LB + 1, LC + 1, LD>(dst, SI, SJ, SK, SL, init, c00, c00p, b10, b01, b00, abx, cdx);
            else if constexpr (LD > 0) fill_2d_smem<LA + 1, LB + 1, LD, LC + 1>(dst, SI, SJ, SL, SK, init, c00, c00p, b10, b01, b00, abx, -cdx);
          } else {
            if (!swk) fill_2d_smem<LB + 1, LA + 1, LC + 1, LD>(dst, SJ, SI, SK, SL, init, c00, c00p, b10, b01, b00, -abx, cdx);
            else if constexpr (LD > 0) fill_2d_smem<LB + 1, LA + 1, LD, LC + 1>(dst, SJ, SI, SL, SK, init, c00, c00p, b10, b01, b00, -abx, -cdx);
          }
        }
        __syncwarp();
        phase2(S, i, ea2, eb2, ec2, false);
      }
    }

    phase3(i);
  }

  } else {
  // ---- paired phase 1 (coop_kernel.cuh): half-warp h builds item h -- a primitive quartet (bra pair, bra primitive pair, ket
  // primitive pair) of the task -- into slab h; the slabs are consumed one after the other, a quartet ends with its phase 3.
  const int h = lane >> 4, hl = lane & 15;
  const int p_root = hl / 3, p_axis = hl - 3 * p_root;
  const bool p_fill = hl < 3 * N;
  const unsigned team = ((1u << (3 * N)) - 1u) << (16 * h);
  double* Sh = S + h * Tr::BASE;
  const int nkb = bp.npp, nkk = kp.npp;
  int i0 = i_begin;
  while (i0 < i_end && j >= w.ket_count[i0]) ++i0;
  int kb0 = 0, kk0 = 0;
  while (i0 < i_end) {
    int i1 = i0, kb1 = kb0, kk1 = kk0 + 1;   // second item: the next primitive quartet of the task
    if (kk1 == nkk) { kk1 = 0; if (++kb1 == nkb) { kb1 = 0; ++i1; while (i1 < i_end && j >= w.ket_count[i1]) ++i1; } }
    const int mi = h ? i1 : i0, mkb = h ? kb1 : kb0, mkk = h ? kk1 : kk0;
    if (p_fill && mi < i_end) {
      double f = bp.geom[6 * bp.stride + mi] * wket;
      if (w.same && mi == j) f *= 0.5;
      double A[3], AB[3];
#pragma unroll
      for (int x = 0; x < 3; ++x) { A[x] = bp.geom[x * bp.stride + mi]; AB[x] = bp.geom[(3 + x) * bp.stride + mi]; }
      const double p = bp.prim[(mkb * 5 + 0) * bp.stride + mi];
      const double P[3] = {bp.prim[(mkb * 5 + 1) * bp.stride + mi], bp.prim[(mkb * 5 + 2) * bp.stride + mi], bp.prim[(mkb * 5 + 3) * bp.stride + mi]};
      const double Kab = bp.prim[(mkb * 5 + 4) * bp.stride + mi];
      bool swb;   // build on B when P is nearer to B (the raised index of B is always transferred)
      {
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
      const double xx = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
      double u, wt;
      rys_root_team<N>(xx, w.rys, p_root, p_axis, 16 * h, team, u, wt);
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
      const double init = ax == 2 ? f * Kab * Kcd * sqrt(rpq) * wt : 1.0;
      double* dst = Sh + (ax * N + p_root) * G2;
      if (!swb) {
        if (!swk) fill_2d_smem<LA + 1, LB + 1, LC + 1, LD>(dst, SI, SJ, SK, SL, init, c00, c00p, b10, b01, b00, abx, cdx);
        else if constexpr (LD > 0) fill_2d_smem<LA + 1, LB + 1, LD, LC + 1>(dst, SI, SJ, SL, SK, init, c00, c00p, b10, b01, b00, abx, -cdx);
      } else {
        if (!swk) fill_2d_smem<LB + 1, LA + 1, LC + 1, LD>(dst, SJ, SI, SK, SL, init, c00, c00p, b10, b01, b00, -abx, cdx);
        else if constexpr (LD > 0) fill_2d_smem<LB + 1, LA + 1, LD, LC + 1>(dst, SJ, SI, SL, SK, init, c00, c00p, b10, b01, b00, -abx, -cdx);
      }
    }
    __syncwarp();
    // dual phase 2: both items at once, one per half-warp, when they belong to one quartet or when every quartet is a single
    // primitive quartet (then each half-warp holds the sums of its own quartet and phase 3 runs by halves)
    const bool both = Tr::DUAL && i1 < i_end && (i0 == i1 || nkb * nkk == 1);
#pragma unroll 1
    for (int t = 0; t < 2; ++t) {   // (not unrolled: one copy of the phase 2 and phase 3 code)
      const int ti = both ? mi : t ? i1 : i0, tkb = both ? mkb : t ? kb1 : kb0, tkk = both ? mkk : t ? kk1 : kk0;
      if (ti >= i_end) break;
      if constexpr (EM != 0) { if (tkb == 0 && tkk == 0) stage(ti); }   // first primitive quartet of a quartet: its density blocks
      const double ea2 = 2.0 * bp.aexp[(tkb * 2 + 0) * bp.stride + ti], eb2 = 2.0 * bp.aexp[(tkb * 2 + 1) * bp.stride + ti];
      const double ec2 = 2.0 * kp.aexp[(tkk * 2 + 0) * kp.stride + j];
      phase2(S + (both ? h : t) * Tr::BASE, ti, ea2, eb2, ec2, both);
      if constexpr (Tr::DUAL) {
        if (both) {
          __syncwarp();   // slab 1 has been read too: the sums may be staged over both slabs
          if (i0 != i1) phase3_halves(i0, i1);
          else if (kb1 == nkb - 1 && kk1 == nkk - 1) phase3(i0);
          break;
        }
      }
      if (tkb == nkb - 1 && tkk == nkk - 1) phase3(ti);   // slab 0 is dead by now: the lane sums are staged there
    }
    __syncwarp();
    i0 = i1; kb0 = kb1; kk0 = kk1 + 1;   // first item of the next pair
    if (i0 < i_end && kk0 == nkk) { kk0 = 0; if (++kb0 == nkb) { kb0 = 0; ++i0; while (i0 < i_end && j >= w.ket_count[i0]) ++i0; } }
  }
  }
  // ---- task end ----
  if (lane < 18) {
    const int jk = lane / 9, ax = lane % 3;
    const int2 at_cd = kp.atom[j];
    double* gout = jk ? w.gK : w.gJ;
    if (keepC != 0.0) atomic_add(gout + 3 * at_cd.x + ax, keepC);
    if (keepD != 0.0) atomic_add(gout + 3 * at_cd.y + ax, keepD);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// EM = 2, "team": the heaviest classes ((gg|fd) ... (gg|gg): more than 10 000 Cartesian elements; raised slab of all roots up
// to 233 KB).  The block is ONE group of TW warps on one quartet: the elements are dealt over all 32 TW lanes (element
// mode), and the roots are processed in chunks of RCH so that the slab of a chunk fits shared memory -- the roots of the
// quadrature are independent terms of Eq. 1, so a chunk is built (phase 1), consumed (phase 2) and overwritten.
// This replaces the generic thread-per-quartet kernel (86 KB of local memory per thread) for these classes.
template <int LA, int LB, int LC, int LD, int TW>
struct CoopGradTeamTraits {
  static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
  static constexpr int NAB = NA * NB, NCD = NC * ND;
  static constexpr int N = nroots_of(LA + LB + LC + LD + 1);
  static constexpr int SCD = ((LC + 2) * (LD + 1)) | 1, G2 = ((LA + 2) * (LB + 2) * SCD) | 1;
  static constexpr int NDQ = NAB + NA * NC + NA * ND + NB * NC + NB * ND + NCD;   // the six density blocks of the quartet
  static constexpr int BUDGET = 200 * 1024 / 8 - NDQ - 18 * TW;                    // doubles left for the slab
  static constexpr int RCH = (BUDGET / (3 * G2) < N) ? BUDGET / (3 * G2) : N;       // roots per chunk
  static_assert(RCH >= 1, "one root's slab does not fit");
  static constexpr int SLAB2D = 3 * RCH * G2;
  static constexpr int BASE = SLAB2D > TW * 32 * 33 ? SLAB2D : TW * 32 * 33;        // the dead slab stages the warp reductions
  static constexpr int SLAB = BASE + NDQ + 18 * TW;
  static constexpr size_t SMEM = sizeof(double) * SLAB;
  static_assert(SMEM <= 227 * 1024, "slab does not fit");
  static_assert(3 * RCH <= 32 * TW, "one lane per (root, axis) of a chunk");
};

template <int LA, int LB, int LC, int LD, int TW>
__global__ void __launch_bounds__(32 * TW) coop_grad_team_kernel(Work w) {
  using Tr = CoopGradTeamTraits<LA, LB, LC, LD, TW>;
  constexpr int NA = Tr::NA, NB = Tr::NB, NC = Tr::NC, ND = Tr::ND, NAB = Tr::NAB, NCD = Tr::NCD;
  constexpr int N = Tr::N, SCD = Tr::SCD, G2 = Tr::G2, RCH = Tr::RCH, T = 32 * TW;
  constexpr int SK = LD + 1, SJ = SCD, SI = (LB + 2) * SCD;
  extern __shared__ __align__(16) double smem[];
  const int lane = threadIdx.x, wy = threadIdx.y, tid = wy * 32 + lane;
  double* S = smem;
  double* sDab = S + Tr::BASE; double* sDac = sDab + NAB; double* sDad = sDac + NA * NC; double* sDbc = sDad + NA * ND;
  double* sDbd = sDbc + NB * NC; double* sDcd = sDbd + NB * ND; double* part = sDcd + NCD;

  const PairSet& bp = w.bra; const PairSet& kp = w.ket;
  const int blk = blockIdx.x * w.nshard + w.shard;
  if (blk >= w.row_off[w.nrows]) return;
  const int r = find_row_warp(w.row_off, w.nrows, blk, lane);
  const int j = blk - w.row_off[r];                  // one ket pair per block
  const int i_begin = r * w.grad_ch, i_end = min(i_begin + w.grad_ch, bp.npair);
  if (j >= kp.npair) return;
  const int n = w.nao;
  const double* __restrict__ D = w.D;
  double C[3], CD[3];
#pragma unroll
  for (int x = 0; x < 3; ++x) { C[x] = kp.geom[x * kp.stride + j]; CD[x] = kp.geom[(3 + x) * kp.stride + j]; }
  const double wket = kp.geom[6 * kp.stride + j];
  const int c0 = kp.ao[j].x, d0 = kp.ao[j].y;
  for (int cd = tid; cd < NCD; cd += T) sDcd[cd] = D[(long)(c0 + cd / ND) * n + d0 + cd % ND];
  double keepC = 0.0, keepD = 0.0;   // warp 0, lane v < 18

  for (int i = i_begin; i < i_end; ++i) {
    if (j >= w.ket_count[i]) continue;     // block-uniform
    double f = bp.geom[6 * bp.stride + i] * wket;
    if (w.same && i == j) f *= 0.5;
    double A[3], AB[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) { A[x] = bp.geom[x * bp.stride + i]; AB[x] = bp.geom[(3 + x) * bp.stride + i]; }
    const int a0 = bp.ao[i].x, b0 = bp.ao[i].y;
    __syncthreads();
    for (int e = tid; e < NAB; e += T) sDab[e] = D[(long)(a0 + e / NB) * n + b0 + e % NB];
    for (int e = tid; e < NA * NC; e += T) sDac[e] = D[(long)(a0 + e / NC) * n + c0 + e % NC];
    for (int e = tid; e < NA * ND; e += T) sDad[e] = D[(long)(a0 + e / ND) * n + d0 + e % ND];
    for (int e = tid; e < NB * NC; e += T) sDbc[e] = D[(long)(b0 + e / NC) * n + c0 + e % NC];
    for (int e = tid; e < NB * ND; e += T) sDbd[e] = D[(long)(b0 + e / ND) * n + d0 + e % ND];

    double acc[18];
#pragma unroll
    for (int e = 0; e < 18; ++e) acc[e] = 0.0;

    for (int kb = 0; kb < bp.npp; ++kb) {
      const double p = bp.prim[(kb * 5 + 0) * bp.stride + i];
      const double P[3] = {bp.prim[(kb * 5 + 1) * bp.stride + i], bp.prim[(kb * 5 + 2) * bp.stride + i], bp.prim[(kb * 5 + 3) * bp.stride + i]};
      const double Kab = bp.prim[(kb * 5 + 4) * bp.stride + i];
      const double ea2 = 2.0 * bp.aexp[(kb * 2 + 0) * bp.stride + i], eb2 = 2.0 * bp.aexp[(kb * 2 + 1) * bp.stride + i];
      bool swb;
      {
        double da = 0.0, db = 0.0;
#pragma unroll
        for (int x = 0; x < 3; ++x) { const double pa = P[x] - A[x], pb = pa + AB[x]; da += pa * pa; db += pb * pb; }
        swb = db < da;
      }
      for (int kk = 0; kk < kp.npp; ++kk) {
        const double q = kp.prim[(kk * 5 + 0) * kp.stride + j];
        const double Q[3] = {kp.prim[(kk * 5 + 1) * kp.stride + j], kp.prim[(kk * 5 + 2) * kp.stride + j], kp.prim[(kk * 5 + 3) * kp.stride + j]};
        const double Kcd = kp.prim[(kk * 5 + 4) * kp.stride + j];
        const double ec2 = 2.0 * kp.aexp[(kk * 2 + 0) * kp.stride + j];
        bool swk = false;
        if (LD > 0) {
          double dc = 0.0, dd = 0.0;
#pragma unroll
          for (int x = 0; x < 3; ++x) { const double qc = Q[x] - C[x], qd = qc + CD[x]; dc += qc * qc; dd += qd * qd; }
          swk = dd < dc;
        }
        const double rpq = 1.0 / (p + q), rho = p * q * rpq;
        const double PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
        const double xx = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
#pragma unroll 1
        for (int r0 = 0; r0 < N; r0 += RCH) {
          const int nr = min(RCH, N - r0);
          // ---- phase 1: lane (root of the chunk, axis) ----
          __syncthreads();
          if (tid < 3 * nr) {
            const int rl = tid / 3, ax = tid - 3 * rl;
            double u, wt;
            rys_root_one<N>(xx, w.rys, r0 + rl, u, wt);
            const double t2 = u * rpq;
            const double b00 = 0.5 * t2, b10 = (1.0 - q * t2) * 0.5 / p, b01 = (1.0 - p * t2) * 0.5 / q;
            const double pa = (ax == 0 ? P[0] - A[0] : ax == 1 ? P[1] - A[1] : P[2] - A[2]);
            const double qc = (ax == 0 ? Q[0] - C[0] : ax == 1 ? Q[1] - C[1] : Q[2] - C[2]);
            const double pqx = (ax == 0 ? PQ[0] : ax == 1 ? PQ[1] : PQ[2]);
            const double abx = (ax == 0 ? AB[0] : ax == 1 ? AB[1] : AB[2]);
            const double cdx = (ax == 0 ? CD[0] : ax == 1 ? CD[1] : CD[2]);
            const double c00 = pa + (swb ? abx : 0.0) - q * t2 * pqx;
            const double c00p = qc + (swk ? cdx : 0.0) + p * t2 * pqx;
            const double init = ax == 2 ? f * Kab * Kcd * sqrt(rpq) * wt : 1.0;
            double* dst = S + (ax * RCH + rl) * G2;
            if (!swb) {
              if (!swk) fill_2d_smem<LA + 1, LB + 1, LC + 1, LD>(dst, SI, SJ, SK, 1, init, c00, c00p, b10, b01, b00, abx, cdx);
              else if constexpr (LD > 0) fill_2d_smem<LA + 1, LB + 1, LD, LC + 1>(dst, SI, SJ, 1, SK, init, c00, c00p, b10, b01, b00, abx, -cdx);
            } else {
              if (!swk) fill_2d_smem<LB + 1, LA + 1, LC + 1, LD>(dst, SJ, SI, SK, 1, init, c00, c00p, b10, b01, b00, -abx, cdx);
              else if constexpr (LD > 0) fill_2d_smem<LB + 1, LA + 1, LD, LC + 1>(dst, SJ, SI, 1, SK, init, c00, c00p, b10, b01, b00, -abx, -cdx);
            }
          }
          __syncthreads();
          // ---- phase 2: the Cartesian elements dealt over all lanes of the block ----
#pragma unroll 1
          for (int e = tid; e < NAB * NCD; e += T) {
            const int id = e % ND, t1 = e / ND, ic = t1 % NC, t2 = t1 / NC, ib = t2 % NB, ia = t2 / NB;
            int ax, ay, az, bx, by, bz, cx, cy, cz, dx, dy, dz;
            cart_powers(LA, ia, ax, ay, az); cart_powers(LB, ib, bx, by, bz); cart_powers(LC, ic, cx, cy, cz); cart_powers(LD, id, dx, dy, dz);
            const double pj = sDab[ia * NB + ib] * sDcd[ic * ND + id];
            const double pk = fma(sDac[ia * NC + ic], sDbd[ib * ND + id], sDad[ia * ND + id] * sDbc[ib * NC + ic]);
            const int ox = ax * SI + bx * SJ + cx * SK + dx, oy = ay * SI + by * SJ + cy * SK + dy + RCH * G2, oz = az * SI + bz * SJ + cz * SK + dz + 2 * RCH * G2;
            const int lax = ax > 0 ? -SI : 0, lay = ay > 0 ? -SI : 0, laz = az > 0 ? -SI : 0;
            const int lbx = bx > 0 ? -SJ : 0, lby = by > 0 ? -SJ : 0, lbz = bz > 0 ? -SJ : 0;
            const int lcx = cx > 0 ? -SK : 0, lcy = cy > 0 ? -SK : 0, lcz = cz > 0 ? -SK : 0;
            const double fax = ax, fay = ay, faz = az, fbx = bx, fby = by, fbz = bz, fcx = cx, fcy = cy, fcz = cz;
#pragma unroll 1
            for (int rt = 0; rt < nr; ++rt) {
              const double* X = S + ox + rt * G2;
              const double* Y = S + oy + rt * G2;
              const double* Z = S + oz + rt * G2;
              const double vx = X[0], vy = Y[0], vz = Z[0];
              const double oyz = vy * vz, oxz = vx * vz, oxy = vx * vy;
              const double dAx = fma(ea2, X[SI], -fax * X[lax]), dAy = fma(ea2, Y[SI], -fay * Y[lay]), dAz = fma(ea2, Z[SI], -faz * Z[laz]);
              const double dBx = fma(eb2, X[SJ], -fbx * X[lbx]), dBy = fma(eb2, Y[SJ], -fby * Y[lby]), dBz = fma(eb2, Z[SJ], -fbz * Z[lbz]);
              const double dCx = fma(ec2, X[SK], -fcx * X[lcx]), dCy = fma(ec2, Y[SK], -fcy * Y[lcy]), dCz = fma(ec2, Z[SK], -fcz * Z[lcz]);
              const double jx = pj * oyz, jy = pj * oxz, jz = pj * oxy;
              const double kx = pk * oyz, ky = pk * oxz, kz = pk * oxy;
              acc[0] = fma(dAx, jx, acc[0]); acc[1] = fma(dAy, jy, acc[1]); acc[2] = fma(dAz, jz, acc[2]);
              acc[3] = fma(dBx, jx, acc[3]); acc[4] = fma(dBy, jy, acc[4]); acc[5] = fma(dBz, jz, acc[5]);
              acc[6] = fma(dCx, jx, acc[6]); acc[7] = fma(dCy, jy, acc[7]); acc[8] = fma(dCz, jz, acc[8]);
              acc[9] = fma(dAx, kx, acc[9]); acc[10] = fma(dAy, ky, acc[10]); acc[11] = fma(dAz, kz, acc[11]);
              acc[12] = fma(dBx, kx, acc[12]); acc[13] = fma(dBy, ky, acc[13]); acc[14] = fma(dBz, kz, acc[14]);
              acc[15] = fma(dCx, kx, acc[15]); acc[16] = fma(dCy, ky, acc[16]); acc[17] = fma(dCz, kz, acc[17]);
            }
          }
        }
      }
    }
    // ---- phase 3: sum over the lanes of each warp through the dead slab, then over the warps ----
#pragma unroll
    for (int e = 0; e < 9; ++e) { acc[e] *= 4.0; acc[9 + e] *= 2.0; }
    __syncthreads();
    if (lane < 18) part[wy * 18 + lane] = 0.0;
    warp_reduce_values<18, false>(acc, S + wy * (32 * 33), lane, [&](int v, int, double sum) { part[wy * 18 + v] = sum; });
    __syncthreads();
    if (wy == 0 && lane < 18) {
      double sum = 0.0;
#pragma unroll
      for (int ww = 0; ww < TW; ++ww) sum += part[ww * 18 + lane];
      const int2 at_ab = bp.atom[i];
      const int jk = lane / 9, ce = (lane % 9) / 3, ax = lane % 3;
      if (ce < 2) atomic_add((jk ? w.gK : w.gJ) + 3 * (ce == 0 ? at_ab.x : at_ab.y) + ax, sum);
      else keepC += sum;
      keepD -= sum;
    }
  }
  if (wy == 0 && lane < 18) {
    const int jk = lane / 9, ax = lane % 3;
    const int2 at_cd = kp.atom[j];
    double* gout = jk ? w.gK : w.gJ;
    if (keepC != 0.0) atomic_add(gout + 3 * at_cd.x + ax, keepC);
    if (keepD != 0.0) atomic_add(gout + 3 * at_cd.y + ax, keepD);
  }
}

template <int LA, int LB, int LC, int LD, int WARPS, int EM>
cudaError_t launch_coop_grad(const Work& w, int nblocks_dense, cudaStream_t s) {
  const int grid = (nblocks_dense + w.nshard - 1) / w.nshard;
  if (grid <= 0) return cudaSuccess;
  static bool attr_set = false;
  if constexpr (EM == 2) {
    using Tr = CoopGradTeamTraits<LA, LB, LC, LD, WARPS>;
    if (!attr_set) {
      cudaError_t e = cudaFuncSetAttribute(coop_grad_team_kernel<LA, LB, LC, LD, WARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tr::SMEM);
      if (e != cudaSuccess) return e;
      attr_set = true;
    }
    coop_grad_team_kernel<LA, LB, LC, LD, WARPS><<<grid, dim3(32, WARPS), Tr::SMEM, s>>>(w);
  } else {
    using Tr = CoopGradTraits<LA, LB, LC, LD, WARPS, EM>;
    if (!attr_set) {
      cudaError_t e = cudaFuncSetAttribute(coop_grad_kernel<LA, LB, LC, LD, WARPS, EM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tr::SMEM);
      if (e != cudaSuccess) return e;
      attr_set = true;
    }
    coop_grad_kernel<LA, LB, LC, LD, WARPS, EM><<<grid, dim3(32, WARPS), Tr::SMEM, s>>>(w);
  }
  return cudaGetLastError();
}

}  // namespace eri
