// launch.h -- host-callable launchers of the kernel translation units of liberi_b200 (internal, not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <string>
#include <vector>
#include "../../include/eri.h"
#include "eri_dev.cuh"

namespace eri {

// generic kernels: block = (GENERIC_BJ ket pairs) x (GENERIC_BI bra pairs), one thread per quartet
constexpr int GENERIC_BJ = 32, GENERIC_BI = 4;
constexpr int GENERIC_GRAD_BJ = 32, GENERIC_GRAD_BI = 4;

cudaError_t launch_generic_jk(const Work& w, int nblocks_dense, cudaStream_t s);
cudaError_t launch_generic_store(const Work& w, double* out, const long long* off, long stride, cudaStream_t s);   // element e of item t at out[off[t] + e * stride]
cudaError_t launch_generic_grad(const Work& w, int nblocks_dense, cudaStream_t s);

// tuned kernels: a launcher per l-class; returns false in `*handled` when the class has no tuned kernel.
struct TunedInfo { int kind; int BI, BJ; int TQ; };   // kind: 1 register-unrolled, 2 cooperative, 3 tile; tile shape for dense mode
// tile family (kind 3, dense mode only): threads per quartet TQ and bra rows per block BI of the class, false if not served
bool tile_jk_info(int la, int lb, int lc, int ld, TunedInfo* info);
cudaError_t launch_tile_jk_class(const Work& w, int nblocks_dense, cudaStream_t s);
bool tuned_jk_info(int la, int lb, int lc, int ld, int npp_bra, int npp_ket, TunedInfo* info);
cudaError_t launch_tuned_jk(const Work& w, int nblocks_dense, cudaStream_t s);
bool tuned_grad_info(int la, int lb, int lc, int ld, int npp_bra, int npp_ket, TunedInfo* info);
cudaError_t launch_tuned_grad(const Work& w, int nblocks_dense, cudaStream_t s);
// cooperative gradient kernel (kind 2, dense mode): info->BI x info->BJ = bra pairs per task x ket pairs per block
bool coop_grad_info(int la, int lb, int lc, int ld, TunedInfo* info);
cudaError_t launch_coop_grad_class(const Work& w, int nblocks_dense, cudaStream_t s);
// primitive-parallel gradient kernel (kind 4, dense mode, pp_grad.cuh): same task shape, lanes own primitive quartets
bool pp_grad_info(int la, int lb, int lc, int ld, TunedInfo* info);
cudaError_t launch_pp_grad_class(const Work& w, int nblocks_dense, cudaStream_t s);

void tuned_catalog(std::vector<std::string>& out);   // "family la lb lc ld" of every tuned instantiation

// transform.cu
cudaError_t upload_c2s(const double* tables /*host, concatenated ns(l) x nc(l), l = 0..LMAX*/);
struct ShellMap {          // device arrays describing the AO layout
  const int* sh_l; const int* sh_sph; const int* sh_cart;   // per shell
  const int* sph2sh; const int* cart2sh;                    // per AO
  int nshell, nao, nao_cart;
};
cudaError_t launch_sph2cart(const ShellMap& m, const double* Dsph, double* Dcart, cudaStream_t s);
// out = T (alpha * (M + M^T if sym else M)) T^T
cudaError_t launch_cart2sph(const ShellMap& m, const double* Mcart, double* Msph, double alpha, int sym, cudaStream_t s);
// spherical blocks from Cartesian blocks: quartet t has shells q4[4t..4t+3], Cartesian block at cart + coff[t], output at out + ooff[t]
cudaError_t launch_block_c2s(const ShellMap& m, const int* q4, int n, const double* cart, const long long* coff,
                             double* out, const long long* ooff, cudaStream_t s);
// Q[t] = sqrt(max_{s,t'} |(s t'|s t')|) over spherical components from the Cartesian block (ab|ab) [nab][nab], element-major:
// element e of pair t at cart[e * n + t]
cudaError_t launch_schwarz_diag(int la, int lb, int n, long stride, const double* cart, double* Q, cudaStream_t s);   // element e of pair t at cart[e * stride + t]
cudaError_t launch_fold_partials(double* cart, long nelem, int m, int split, cudaStream_t s);   // sums the `split` partial blocks of the Schwarz pass into the first
cudaError_t launch_diag_list(int2* list, long long* off, int start, int m, int split, cudaStream_t s);
// density-weighted screening (transform.cu): shell-group sub-block maxima of |D|, then per unit the effective threshold,
// the per-call kept ket counts and the number of quartets that pass
struct DscreenUnit { const double* qb; const double* qk; const int* count; int* count_dyn; int nbra; int g[4]; };
cudaError_t launch_group_max(const double* D, int nao, const int* ao_group, int ng, unsigned long long* pmax, cudaStream_t s);
// the same maxima as doubles in P[ng*ng], accumulators in a file-scope device array (no allocation; ng <= ERI_NOALLOC_MAX_GROUPS)
cudaError_t launch_group_max_noalloc(const double* D, int nao, const int* ao_group, int ng, double* P, cudaStream_t s);
cudaError_t launch_dscreen(const DscreenUnit* units, int nunits, int max_nbra, const unsigned long long* pmax, int ng, double tau,
                           double* thr_eff, unsigned long long* kept, cudaStream_t s);
// primitive-pair records of the pairs (sa[i], sb[i]) from the shell data on the device (plan creation); arrays zeroed by the caller
cudaError_t launch_build_pairs(const eri_shell_t* sh, const eri_prim_t* pr, const double* xyz, const int* cart_off, const int* sa, const int* sb,
                               int n, int Kb, int npp, long st, double kfac /* sqrt(2) pi^(5/4) */, double* prim, double* geom, double* aexp, int2* ao, int2* atom, cudaStream_t s);
// dst[r * dstride + i] = src[r * sstride + idx[i]], r < rows, i < n (SoA pair records); dst[i] = src[idx[i]] for the int2 arrays
cudaError_t launch_gather_rows(const double* src, double* dst, const int* idx, int n, int rows, long sstride, long dstride, cudaStream_t s);
cudaError_t launch_gather_int2(const int2* src, int2* dst, const int* idx, int n, cudaStream_t s);
cudaError_t launch_rys_diag(int N, const double* rys, const double* x, int n, double* u, double* w, cudaStream_t s);
cudaError_t launch_fp64_peak(double* sink, int iters, int blocks, cudaStream_t s);

}  // namespace eri
