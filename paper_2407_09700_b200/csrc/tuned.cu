// tuned.cu -- dispatch table of the per-class tuned kernels: register family (reg_g*.cu), cooperative family (coop_*.cu).
#include <cstdio>
#include <string>
#include <vector>
#include "launch.h"
#include "reg_classes.h"
#include "coop_classes.h"
#include "tile_classes.h"
#include "tile_grad_classes.h"
#include "coop_grad_classes.h"
#include "pp_grad_classes.h"

namespace eri {

bool launch_reg_group0(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err);
bool launch_reg_group1(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err);
bool launch_reg_group2(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err);
bool launch_reg_group3(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err);

#define DECL(g) bool launch_coop_group##g(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err);
DECL(0) DECL(1) DECL(2) DECL(3) DECL(4) DECL(5) DECL(6) DECL(7)
#undef DECL
static_assert(COOP_NGROUPS == 8, "tuned.cu lists eight cooperative groups");
#define COOP_ALL(X) COOP_GROUP0(X) COOP_GROUP1(X) COOP_GROUP2(X) COOP_GROUP3(X) COOP_GROUP4(X) COOP_GROUP5(X) COOP_GROUP6(X) COOP_GROUP7(X)

// warps per quartet of a cooperative class, 0 if the class is not served
static int coop_tw(int key) {
  switch (key) {
#define X(a, b, c, d, tw, nch) case a * 1000 + b * 100 + c * 10 + d: return tw;
    COOP_ALL(X)
#undef X
    default: return 0;
  }
}

static bool is_reg_class(int key) {
  switch (key) {
#define X(a, b, c, d) case a * 1000 + b * 100 + c * 10 + d:
    REG_GROUP0(X) REG_GROUP1(X) REG_GROUP2(X) REG_GROUP3(X)
#undef X
      return true;
    default: return false;
  }
}

bool tuned_jk_info(int la, int lb, int lc, int ld, int, int, TunedInfo* info) {
  const int key = la * 1000 + lb * 100 + lc * 10 + ld;
  if (is_reg_class(key)) { info->kind = 1; info->BI = 4; info->BJ = 32; return true; }
  if (const int tw = coop_tw(key)) { info->kind = 2; info->BI = 16; info->BJ = tw > 4 ? 1 : 4 / tw; return true; }   // COOP_CH bra pairs x (max(COOP_WARPS, TW) / TW) ket pairs
  return false;
}

cudaError_t launch_tuned_jk(const Work& w, int nblocks, cudaStream_t s) {
  const int key = w.bra.la * 1000 + w.bra.lb * 100 + w.ket.la * 10 + w.ket.lb;
  cudaError_t err = cudaErrorNotSupported;
  if (launch_reg_group0(key, w, nblocks, s, &err)) return err;
  if (launch_reg_group1(key, w, nblocks, s, &err)) return err;
  if (launch_reg_group2(key, w, nblocks, s, &err)) return err;
  if (launch_reg_group3(key, w, nblocks, s, &err)) return err;
#define TRY(g) if (launch_coop_group##g(key, w, nblocks, s, &err)) return err;
  TRY(0) TRY(1) TRY(2) TRY(3) TRY(4) TRY(5) TRY(6) TRY(7)
#undef TRY
  return cudaErrorNotSupported;
}

// ---- tile family (dense mode only) ----
#define DECL(g) bool launch_tile_group##g(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err);
DECL(0) DECL(1) DECL(2) DECL(3) DECL(4) DECL(5) DECL(6) DECL(7)
#undef DECL
static_assert(TILE_NGROUPS == 8, "tuned.cu lists eight tile groups");
#define TILE_ALL(X) TILE_GROUP0(X) TILE_GROUP1(X) TILE_GROUP2(X) TILE_GROUP3(X) TILE_GROUP4(X) TILE_GROUP5(X) TILE_GROUP6(X) TILE_GROUP7(X)

bool tile_jk_info(int la, int lb, int lc, int ld, TunedInfo* info) {
  switch (la * 1000 + lb * 100 + lc * 10 + ld) {
#define X(a, b, c, d, tq, bi) case a * 1000 + b * 100 + c * 10 + d: info->kind = 3; info->TQ = tq; info->BI = bi; info->BJ = 32; return true;
    TILE_ALL(X)
#undef X
    default: return false;
  }
}

cudaError_t launch_tile_jk_class(const Work& w, int nblocks, cudaStream_t s) {
  const int key = w.bra.la * 1000 + w.bra.lb * 100 + w.ket.la * 10 + w.ket.lb;
  cudaError_t err = cudaErrorNotSupported;
#define TRY(g) if (launch_tile_group##g(key, w, nblocks, s, &err)) return err;
  TRY(0) TRY(1) TRY(2) TRY(3) TRY(4) TRY(5) TRY(6) TRY(7)
#undef TRY
  return cudaErrorNotSupported;
}

// ---- tile family, gradient (dense mode only) ----
#define DECL(g) bool launch_tgrad_group##g(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err);
DECL(0) DECL(1) DECL(2) DECL(3) DECL(4) DECL(5) DECL(6) DECL(7)
#undef DECL
static_assert(TGRAD_NGROUPS == 8, "tuned.cu lists eight tile gradient groups");
#define TGRAD_ALL(X) TGRAD_GROUP0(X) TGRAD_GROUP1(X) TGRAD_GROUP2(X) TGRAD_GROUP3(X) TGRAD_GROUP4(X) TGRAD_GROUP5(X) TGRAD_GROUP6(X) TGRAD_GROUP7(X)

#define DECL(g) bool launch_cgrad_group##g(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err);
DECL(0) DECL(1) DECL(2) DECL(3) DECL(4) DECL(5) DECL(6) DECL(7)
#undef DECL
static_assert(CGRAD_NGROUPS == 8, "tuned.cu lists eight cooperative gradient groups");
#define CGRAD_ALL(X) CGRAD_GROUP0(X) CGRAD_GROUP1(X) CGRAD_GROUP2(X) CGRAD_GROUP3(X) CGRAD_GROUP4(X) CGRAD_GROUP5(X) CGRAD_GROUP6(X) CGRAD_GROUP7(X)

// cooperative gradient kernel (kind 2): Schwarz-sorted pair sets, task = 16 bra pairs x 1 ket pair, `warps` ket pairs per block
bool coop_grad_info(int la, int lb, int lc, int ld, TunedInfo* info) {
  switch (la * 1000 + lb * 100 + lc * 10 + ld) {
#define X(a, b, c, d, wp, em) case a * 1000 + b * 100 + c * 10 + d: info->kind = 2; info->TQ = 1; info->BI = 16; info->BJ = (em == 2 ? 1 : wp); return true;   // EM = 2: the block is one team on one ket pair
    CGRAD_ALL(X)
#undef X
    default: return false;
  }
}

cudaError_t launch_coop_grad_class(const Work& w, int nblocks, cudaStream_t s) {
  const int key = w.bra.la * 1000 + w.bra.lb * 100 + w.ket.la * 10 + w.ket.lb;
  cudaError_t err = cudaErrorNotSupported;
#define TRY(g) if (launch_cgrad_group##g(key, w, nblocks, s, &err)) return err;
  TRY(0) TRY(1) TRY(2) TRY(3) TRY(4) TRY(5) TRY(6) TRY(7)
#undef TRY
  return cudaErrorNotSupported;
}

// ---- primitive-parallel gradient kernel (kernel_grad 4, dense mode): task shape of the cooperative gradient kernel, PGRAD_WARPS ket pairs per block ----
bool launch_pgrad_group0(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err);
bool launch_pgrad_group1(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err);
static_assert(PGRAD_NGROUPS == 2, "tuned.cu lists two primitive-parallel gradient groups");

bool pp_grad_info(int la, int lb, int lc, int ld, TunedInfo* info) {
  switch (la * 1000 + lb * 100 + lc * 10 + ld) {
#define X(a, b, c, d) case a * 1000 + b * 100 + c * 10 + d:
    PGRAD_GROUP0(X) PGRAD_GROUP1(X)
#undef X
      info->kind = 4; info->TQ = 1; info->BI = 16; info->BJ = 4; return true;   // BJ = PGRAD_WARPS (pp_grad.cuh)
    default: return false;
  }
}

cudaError_t launch_pp_grad_class(const Work& w, int nblocks, cudaStream_t s) {
  const int key = w.bra.la * 1000 + w.bra.lb * 100 + w.ket.la * 10 + w.ket.lb;
  cudaError_t err = cudaErrorNotSupported;
  if (launch_pgrad_group0(key, w, nblocks, s, &err)) return err;
  if (launch_pgrad_group1(key, w, nblocks, s, &err)) return err;
  return cudaErrorNotSupported;
}

bool tuned_grad_info(int la, int lb, int lc, int ld, int npp_bra, int npp_ket, TunedInfo* info) {
  // few quartets with 24 primitive ket pairs (K = 3 x 8) fill the tile's 32 ket slots badly; measured on cfg4: faster on the cooperative kernel
  // for the (x|ps) classes, slower for (x|ss) and for the contracted (ds|pp), (pp|pp) units (profiles/r01f_cfg4.md)
  if (lc >= 1 && npp_ket >= 24) return false;
  switch (la * 1000 + lb * 100 + lc * 10 + ld) {
#define X(a, b, c, d, bi, mode) case a * 1000 + b * 100 + c * 10 + d: info->kind = 3; info->TQ = 1; info->BI = bi; info->BJ = 32; return true;
    TGRAD_ALL(X)
#undef X
    default: return false;
  }
}

cudaError_t launch_tuned_grad(const Work& w, int nblocks, cudaStream_t s) {
  const int key = w.bra.la * 1000 + w.bra.lb * 100 + w.ket.la * 10 + w.ket.lb;
  cudaError_t err = cudaErrorNotSupported;
#define TRY(g) if (launch_tgrad_group##g(key, w, nblocks, s, &err)) return err;
  TRY(0) TRY(1) TRY(2) TRY(3) TRY(4) TRY(5) TRY(6) TRY(7)
#undef TRY
  return cudaErrorNotSupported;
}

// every (family, class) instantiation the library holds, "family la lb lc ld" (eri_kernel_catalog)
void tuned_catalog(std::vector<std::string>& out) {
  auto add = [&](const char* fam, int a, int b, int c, int d) {
    char buf[64]; snprintf(buf, sizeof buf, "%s %d %d %d %d", fam, a, b, c, d); out.push_back(buf);
  };
#define X(a, b, c, d) add("reg", a, b, c, d);
  REG_GROUP0(X) REG_GROUP1(X) REG_GROUP2(X) REG_GROUP3(X)
#undef X
#define X(a, b, c, d, tw, nch) add("coop", a, b, c, d);
  COOP_ALL(X)
#undef X
#define X(a, b, c, d, tq, bi) add("tile", a, b, c, d);
  TILE_ALL(X)
#undef X
#define X(a, b, c, d, bi, mode) add("tgrad", a, b, c, d);
  TGRAD_ALL(X)
#undef X
#define X(a, b, c, d, wp, em) add("cgrad", a, b, c, d);
  CGRAD_ALL(X)
#undef X
#define X(a, b, c, d) add("pgrad", a, b, c, d);
  PGRAD_GROUP0(X) PGRAD_GROUP1(X)
#undef X
}

}  // namespace eri
