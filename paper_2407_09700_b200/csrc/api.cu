// api.cu -- host side of liberi_b200: the C ABI of include/eri.h, the plan builder (shell grouping, pair sets,
// Schwarz bounds, Schwarz-sorted task lists; Algorithm 1 lines 1-8) and kernel dispatch.
// Product code: there is no CPU fallback and nothing from oracle/ is used here.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <deque>
#include <map>
#include <memory>
#include <mutex>
#include <new>
#include <set>
#include <string>
#include <thread>
#include <vector>

#include "../../include/eri.h"
#include "eri_dev.cuh"
#include "launch.h"
#include "rys_tables.inc"

namespace eri {
namespace {

thread_local std::string g_err;

int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
  g_err = buf;
  return code;
}
#define CK(call)                                                                                       \
  do {                                                                                                 \
    cudaError_t e_ = (call);                                                                           \
    if (e_ != cudaSuccess) return fail(e_ == cudaErrorMemoryAllocation ? ERI_ERR_NOMEM : ERI_ERR_CUDA, \
                                       "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
  } while (0)
#define CKI(call) do { int r_ = (call); if (r_ != ERI_OK) return r_; } while (0)

// Device allocations go through the stream-ordered allocator on a private stream with the pool's release threshold lifted:
// a plan makes some thousand small allocations (pair sets, row tables), and cudaMalloc / cudaFree (each an implicit device
// synchronisation) were a third of plan creation (profiles/r02_plan.md).  alloc() waits for its own allocation, so the
// pointer is usable on any stream; release() is ordered on the private stream only, so every owner synchronises the streams
// that used the buffer before it lets go of it (plan creation does; eri_plan_destroy synchronises the device first).
cudaStream_t g_alloc_stream = nullptr;
cudaError_t alloc_stream(cudaStream_t* out) {
  static std::mutex mu;
  std::lock_guard<std::mutex> lk(mu);
  if (!g_alloc_stream) {
    cudaError_t e = cudaStreamCreateWithFlags(&g_alloc_stream, cudaStreamNonBlocking);
    if (e != cudaSuccess) return e;
    int dev = 0; cudaMemPool_t pool = nullptr;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
      unsigned long long keep = ~0ull;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
  }
  *out = g_alloc_stream;
  return cudaSuccess;
}

template <class T>
struct Dev {   // owning device array
  T* p = nullptr; size_t n = 0;
  Dev() = default;
  Dev(const Dev&) = delete; Dev& operator=(const Dev&) = delete;
  Dev(Dev&& o) noexcept : p(o.p), n(o.n) { o.p = nullptr; o.n = 0; }
  Dev& operator=(Dev&& o) noexcept { if (this != &o) { release(); p = o.p; n = o.n; o.p = nullptr; o.n = 0; } return *this; }
  ~Dev() { release(); }
  void release() { if (p) { if (g_alloc_stream) cudaFreeAsync(p, g_alloc_stream); else cudaFree(p); } p = nullptr; n = 0; }
  cudaError_t alloc(size_t count) {
    release();
    if (count == 0) return cudaSuccess;
    cudaStream_t as = nullptr;
    cudaError_t e = alloc_stream(&as);
    if (e != cudaSuccess) return e;
    e = cudaMallocAsync(&p, count * sizeof(T), as);
    if (e != cudaSuccess) { p = nullptr; return e; }
    n = count;
    return cudaStreamSynchronize(as);
  }
  // the copy runs on the allocator's private stream and is complete on return: the data can then be used on any stream, and
  // uploads never wait for (or serialise with) kernels queued on the caller's stream, e.g. the Schwarz pass of plan creation
  cudaError_t upload(const std::vector<T>& h, cudaStream_t /*unused*/) {
    cudaError_t e = alloc(h.size());
    if (e != cudaSuccess || h.empty()) return e;
    e = cudaMemcpyAsync(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, g_alloc_stream);
    if (e != cudaSuccess) return e;
    return cudaStreamSynchronize(g_alloc_stream);
  }
};

// ---- process-wide read-only device data ---------------------------------------------------------------------
// The library binds to the device that is current at its first compute call: the Rys buffer, the __constant__ c2s table and
// the per-kernel shared-memory attributes live on that device.  Every later entry point checks that the same device is
// current and fails with ERI_ERR_BAD_ARG otherwise (eri.h "Devices"); one process drives one GPU.
std::mutex g_init_mu;
double* g_rys = nullptr;
int g_device = -1;
bool g_c2s_ready = false;
std::vector<double> g_c2s_host[LMAX + 1];

double binom(int n, int k) { if (k < 0 || k > n) return 0.0; double r = 1.0; for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i; return r; }
double fact(int n) { double r = 1.0; for (int i = 2; i <= n; ++i) r *= i; return r; }
int cart_index(int l, int lx, int ly) {  // lx descending, then ly descending
  int idx = 0;
  for (int x = l; x > lx; --x) idx += l - x + 1;
  return idx + (l - lx - ly);
}

// Real solid harmonics, unit-normalised on the sphere, m = -l..l (reading R3): closed formula
//   Y_lm = sqrt((2l+1)/4pi) N_lm sum_{t,u,v} C^{lm}_{tuv} x^{2t+|m|-2(u+v)} y^{2(u+v)} z^{l-2t-|m|}.
void build_c2s(int l, std::vector<double>& T) {
  const int nc = ncart(l), ns = nsph(l);
  T.assign((size_t)ns * nc, 0.0);
  for (int m = -l; m <= l; ++m) {
    const int am = std::abs(m);
    const double Nlm = std::sqrt(2.0 * fact(l + am) * fact(l - am) / (m == 0 ? 2.0 : 1.0)) / (std::pow(2.0, am) * fact(l));
    const double norm = std::sqrt((2 * l + 1) / (4.0 * PI)) * Nlm;
    const int v2min = m < 0 ? 1 : 0;   // 2v runs over v2min, v2min+2, ... <= |m|
    for (int t = 0; t <= (l - am) / 2; ++t)
      for (int u = 0; u <= t; ++u)
        for (int v2 = v2min; v2 <= am; v2 += 2) {
          const int sign_exp = t + (v2 - v2min) / 2;
          const double C = ((sign_exp & 1) ? -1.0 : 1.0) * std::pow(0.25, t) * binom(l, t) * binom(l - t, am + t) * binom(t, u) * binom(am, v2);
          const int ex = 2 * t + am - (2 * u + v2), ey = 2 * u + v2, ez = l - 2 * t - am;
          if (ex < 0 || ey < 0 || ez < 0) continue;
          T[(size_t)(m + l) * nc + cart_index(l, ex, ey)] += norm * C;
        }
  }
}

int ensure_init() {
  std::lock_guard<std::mutex> lk(g_init_mu);
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (g_device >= 0 && dev != g_device)
    return fail(ERI_ERR_BAD_ARG, "liberi_b200 is bound to CUDA device %d (current at its first call) but device %d is current", g_device, dev);
  if (!g_rys) {
    // consistency of the compile-time constants in eri_dev.cuh with the generated table
    static_assert(RYS_NMAX == RYS_NROOTS_MAX, "rys_tables.inc must tabulate N = 1..RYS_NROOTS_MAX");
    for (int N = 1; N <= RYS_NMAX; ++N)
      if (rys_offset(N) != RYS_TABLE_OFFSET_H[N] || rys_xmax(N) != RYS_XMAX_H[N])
        return fail(ERI_ERR_BAD_ARG, "rys_tables.inc does not match eri_dev.cuh (N=%d)", N);
    static_assert(RYS_TABLE_DOUBLES == RYS_TABLE_SIZE, "eri_dev.cuh: RYS_TABLE_DOUBLES must equal RYS_TABLE_SIZE of rys_tables.inc");
    static_assert(RYS2_BASE % 2 == 0, "second table layout must start 16-byte aligned");
    std::vector<double> h(RYS2_BASE + rys2_offset(RYS2_NMAX + 1), 0.0);
    for (int N = 1; N <= RYS_NMAX; ++N) { h[RYS_HDR_XMAX + N] = RYS_XMAX_H[N]; h[RYS_HDR_OFF + N] = RYS_TABLE_OFFSET_H[N]; }
    for (int k = 0; k < RYS_NMAX * (RYS_NMAX + 1) / 2; ++k) { h[RYS_HDR_H2 + k] = RYS_HERM_H2_H[k]; h[RYS_HDR_V + k] = RYS_HERM_V_H[k]; }
    std::memcpy(h.data() + RYS_HDR_SIZE, RYS_TABLE_H, sizeof(double) * RYS_TABLE_SIZE);
    // second layout (eri_dev.cuh "Shared-memory copy"): [interval][value][k], padded interval stride
    for (int N = 1; N <= RYS2_NMAX; ++N)
      for (int iv = 0; iv < rys_nint(N); ++iv)
        for (int k = 0; k < 14; ++k)
          for (int n = 0; n < 2 * N; ++n)
            h[RYS2_BASE + rys2_offset(N) + (size_t)iv * rys2_stride(N) + n * 14 + k] = RYS_TABLE_H[RYS_TABLE_OFFSET_H[N] + iv * (28 * N) + k * 2 * N + n];
    double* d = nullptr;
    CK(cudaMalloc(&d, h.size() * sizeof(double)));
    CK(cudaMemcpy(d, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice));
    g_rys = d;
    g_device = dev;
  }
  if (!g_c2s_ready) {
    std::vector<double> all;
    for (int l = 0; l <= LMAX; ++l) { build_c2s(l, g_c2s_host[l]); all.insert(all.end(), g_c2s_host[l].begin(), g_c2s_host[l].end()); }
    size_t want = 0; for (int l = 0; l <= LMAX; ++l) want += (size_t)nsph(l) * ncart(l);
    if (all.size() != want) return fail(ERI_ERR_BAD_ARG, "internal: c2s table size");
    CK(upload_c2s(all.data()));
    g_c2s_ready = true;
  }
  return ERI_OK;
}

// Host loops of plan creation over a few worker threads (pair records, work units): contiguous ranges, the workers bind to the
// library's device first (a new host thread starts on device 0).  f(lo, hi) returns an eri error code; the first failure wins.
template <class F>
int parallel_ranges(int n, int min_per_thread, F f) {
  const int hw = (int)std::thread::hardware_concurrency();
  const int nt = std::max(1, std::min(std::min(hw > 0 ? hw : 4, 16), n / std::max(1, min_per_thread)));
  if (nt <= 1) return f(0, n);
  std::vector<int> rc(nt, ERI_OK);
  std::vector<std::string> msg(nt);
  std::vector<std::thread> th;
  for (int t = 0; t < nt; ++t)
    th.emplace_back([&, t] {
      if (g_device >= 0) cudaSetDevice(g_device);
      rc[t] = f((int)((long long)n * t / nt), (int)((long long)n * (t + 1) / nt));
      if (rc[t] != ERI_OK) msg[t] = g_err;
    });
  for (auto& x : th) x.join();
  for (int t = 0; t < nt; ++t) if (rc[t] != ERI_OK) { g_err = msg[t]; return rc[t]; }
  return ERI_OK;
}

// ---- basis ----------------------------------------------------------------------------------------------------
struct Group { int l, K; std::vector<int> shells; };

struct Basis {
  std::vector<eri_shell_t> sh; std::vector<eri_prim_t> pr; std::vector<double> xyz;
  int natm = 0, nao = 0, nao_cart = 0;
  std::vector<int> cart_off, group_of;
  std::vector<Group> groups;   // sorted by (l, K)
};

int make_basis(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim, const double* coords, int natm, Basis& b) {
  if (nshell < 0 || nprim < 0 || natm < 0) return fail(ERI_ERR_BAD_ARG, "negative count");
  if ((nshell > 0 && (!shells || !prims || !coords))) return fail(ERI_ERR_BAD_ARG, "null basis pointer");
  b.sh.assign(shells, shells + nshell); b.pr.assign(prims, prims + nprim); b.xyz.assign(coords, coords + 3 * (size_t)natm);
  b.natm = natm; b.nao = 0; b.nao_cart = 0;
  b.cart_off.resize(nshell); b.group_of.resize(nshell);
  std::map<std::pair<int, int>, int> gid;
  for (int s = 0; s < nshell; ++s) {
    const eri_shell_t& S = shells[s];
    if (S.l < 0 || S.l > LMAX) return fail(ERI_ERR_UNSUPPORTED_L, "shell %d: l = %d is outside 0..%d", s, S.l, LMAX);
    if (S.nprim <= 0) return fail(ERI_ERR_BAD_ARG, "shell %d: nprim = %d", s, S.nprim);
    if (S.prim_off < 0 || (long)S.prim_off + S.nprim > nprim) return fail(ERI_ERR_BAD_ARG, "shell %d: primitive range outside prims", s);
    if (S.atom < 0 || S.atom >= natm) return fail(ERI_ERR_BAD_ARG, "shell %d: atom %d outside 0..%d", s, S.atom, natm - 1);
    if (S.ao_off != b.nao) return fail(ERI_ERR_BAD_ARG, "shell %d: ao_off = %d, expected running sum %d", s, S.ao_off, b.nao);
    for (int k = 0; k < S.nprim; ++k) {
      const double e = prims[S.prim_off + k].exp, c = prims[S.prim_off + k].coef;
      if (!(e > 0.0) || !std::isfinite(e) || !std::isfinite(c)) return fail(ERI_ERR_BAD_ARG, "shell %d: bad primitive %d", s, k);
    }
    b.cart_off[s] = b.nao_cart;
    b.nao += nsph(S.l); b.nao_cart += ncart(S.l);
    gid[{S.l, S.nprim}] = 0;
  }
  for (int x = 0; x < 3 * natm; ++x) if (!std::isfinite(coords[x])) return fail(ERI_ERR_BAD_ARG, "non-finite coordinate");
  int g = 0;
  for (auto& kv : gid) { kv.second = g++; b.groups.push_back(Group{kv.first.first, kv.first.second, {}}); }
  for (int s = 0; s < nshell; ++s) { const int id = gid[{shells[s].l, shells[s].nprim}]; b.group_of[s] = id; b.groups[id].shells.push_back(s); }
  return ERI_OK;
}

// ---- pair sets ------------------------------------------------------------------------------------------------
struct PairClass {
  int ga = 0, gb = 0, la = 0, lb = 0, Ka = 0, Kb = 0, npp = 0, npair = 0, stride = 0;
  std::vector<int> sa, sb;       // shell ids, first / second
  std::vector<double> Q, wgt;    // Schwarz factor, pair weight
  Dev<double> prim, geom, aexp, q;
  Dev<int2> ao, atom;
  // tile family: the same pairs in chunks of 32 slots that share the first shell (padding slots have Q = -1);
  // chunks are ordered by decreasing largest Schwarz factor, which is the factor of the chunk's first slot
  std::unique_ptr<PairClass> grouped;
  std::vector<int> src;            // grouped only: index of every slot's pair in the Schwarz-sorted set (padding slots repeat a pair of their half)
  std::vector<double> half_q;      // grouped only: largest Schwarz factor of each half-chunk of 16 slots (sorted by it, descending; -1: padding)
  double fill = 0.0;               // grouped only: valid slots / slots
  double hrr_loss_grad = 1.0;      // the same with lb + 1 quanta (gradient kernels raise the second shell too)
  double hrr_loss = 1.0;           // max over primitive pairs of ((alpha_a + alpha_b) / alpha_a)^lb, see DESIGN.md "HRR direction"
  PairSet view() const {
    PairSet v; v.prim = prim.p; v.geom = geom.p; v.aexp = aexp.p; v.q = q.p; v.ao = ao.p; v.atom = atom.p;
    v.npair = npair; v.stride = stride; v.npp = npp; v.la = la; v.lb = lb; return v;
  }
};

// fills and uploads the SoA arrays of pc from pc.sa/sb/wgt/Q (Q may be empty)
int upload_pair_class(const Basis& b, PairClass& pc, cudaStream_t s) {
  const int n = pc.npair = (int)pc.sa.size();
  pc.stride = (n + 31) / 32 * 32;
  if (n == 0) return ERI_OK;
  const size_t st = pc.stride;
  std::vector<double> prim((size_t)pc.npp * 5 * st, 0.0), geom(7 * st, 0.0), aexp((size_t)pc.npp * 2 * st, 0.0), q(st, 0.0);
  std::vector<int2> ao(st, make_int2(0, 0)), atom(st, make_int2(0, 0));
  const double kfac = std::sqrt(2.0) * std::pow(PI, 1.25);
  parallel_ranges(n, std::max(1, 16384 / pc.npp), [&](int lo_i, int hi_i) {
  for (int i = lo_i; i < hi_i; ++i) {
    const eri_shell_t& A = b.sh[pc.sa[i]]; const eri_shell_t& B = b.sh[pc.sb[i]];
    const double* RA = &b.xyz[3 * A.atom]; const double* RB = &b.xyz[3 * B.atom];
    const double ab[3] = {RA[0] - RB[0], RA[1] - RB[1], RA[2] - RB[2]};
    const double r2 = ab[0] * ab[0] + ab[1] * ab[1] + ab[2] * ab[2];
    for (int x = 0; x < 3; ++x) { geom[x * st + i] = RA[x]; geom[(3 + x) * st + i] = ab[x]; }
    geom[6 * st + i] = pc.wgt.empty() ? 1.0 : pc.wgt[i];
    ao[i] = make_int2(b.cart_off[pc.sa[i]], b.cart_off[pc.sb[i]]);
    atom[i] = make_int2(A.atom, B.atom);
    if (!pc.Q.empty()) q[i] = pc.Q[i];
    int k = 0;
    for (int ka = 0; ka < A.nprim; ++ka)
      for (int kb = 0; kb < B.nprim; ++kb, ++k) {
        const double ea = b.pr[A.prim_off + ka].exp, eb = b.pr[B.prim_off + kb].exp;
        const double ca = b.pr[A.prim_off + ka].coef, cb = b.pr[B.prim_off + kb].coef;
        const double p = ea + eb;
        prim[((size_t)k * 5 + 0) * st + i] = p;
        for (int x = 0; x < 3; ++x) prim[((size_t)k * 5 + 1 + x) * st + i] = (ea * RA[x] + eb * RB[x]) / p;
        prim[((size_t)k * 5 + 4) * st + i] = kfac / p * ca * cb * std::exp(-ea * eb / p * r2);
        aexp[((size_t)k * 2 + 0) * st + i] = ea; aexp[((size_t)k * 2 + 1) * st + i] = eb;
      }
  }
  return (int)ERI_OK; });
  CK(pc.prim.upload(prim, s)); CK(pc.geom.upload(geom, s)); CK(pc.aexp.upload(aexp, s)); CK(pc.q.upload(q, s));
  CK(pc.ao.upload(ao, s)); CK(pc.atom.upload(atom, s));   // complete on return (Dev::upload)
  return ERI_OK;
}

// The records of dst's pairs (dst.sa/sb/wgt/Q filled; pair i of dst is pair idx[i] of src) gathered on the device from src's
// arrays -- bit-identical to upload_pair_class, without rebuilding them on the host and sending them over PCIe a second time.
// Runs on the allocator's private stream and is complete on return, like Dev::upload.
int gather_pair_class(const PairClass& src, const std::vector<int>& idx, PairClass& dst) {
  const int n = dst.npair = (int)idx.size();
  dst.stride = (n + 31) / 32 * 32;
  if (n == 0) return ERI_OK;
  const size_t st = dst.stride;
  CK(dst.prim.alloc((size_t)dst.npp * 5 * st)); CK(dst.geom.alloc(7 * st)); CK(dst.aexp.alloc((size_t)dst.npp * 2 * st));
  CK(dst.ao.alloc(st)); CK(dst.atom.alloc(st));
  Dev<int> idxd;
  CK(idxd.upload(idx, g_alloc_stream));
  std::vector<double> q(st, 0.0);
  for (int i = 0; i < n; ++i) q[i] = dst.Q[i];
  CK(dst.q.upload(q, g_alloc_stream));
  cudaStream_t as = g_alloc_stream;
  CK(cudaMemsetAsync(dst.prim.p, 0, sizeof(double) * dst.prim.n, as)); CK(cudaMemsetAsync(dst.geom.p, 0, sizeof(double) * dst.geom.n, as));
  CK(cudaMemsetAsync(dst.aexp.p, 0, sizeof(double) * dst.aexp.n, as));
  CK(cudaMemsetAsync(dst.ao.p, 0, sizeof(int2) * st, as)); CK(cudaMemsetAsync(dst.atom.p, 0, sizeof(int2) * st, as));
  CK(launch_gather_rows(src.prim.p, dst.prim.p, idxd.p, n, dst.npp * 5, src.stride, st, as));
  CK(launch_gather_rows(src.geom.p, dst.geom.p, idxd.p, n, 7, src.stride, st, as));
  CK(launch_gather_rows(src.aexp.p, dst.aexp.p, idxd.p, n, dst.npp * 2, src.stride, st, as));
  CK(launch_gather_int2(src.ao.p, dst.ao.p, idxd.p, n, as)); CK(launch_gather_int2(src.atom.p, dst.atom.p, idxd.p, n, as));
  CK(cudaStreamSynchronize(as));   // idxd is released on return
  return ERI_OK;
}

// The basis on the device, for building pair records there (dense plans: 9e5 primitive pairs at cfg3 took the host 40 ms to
// build and send; profiles/r02_plan.md)
struct BasisDev { Dev<eri_shell_t> sh; Dev<eri_prim_t> pr; Dev<double> xyz; Dev<int> cart_off; };
int upload_basis(const Basis& b, BasisDev& d, cudaStream_t s) {
  CK(d.sh.upload(b.sh, s)); CK(d.pr.upload(b.pr, s)); CK(d.xyz.upload(b.xyz, s)); CK(d.cart_off.upload(b.cart_off, s));
  return ERI_OK;
}
// as upload_pair_class, the records computed on the device (pc.wgt is the rule 1/2 for a shell with itself, as everywhere)
int build_pair_class_device(const BasisDev& bd, PairClass& pc) {
  const int n = pc.npair = (int)pc.sa.size();
  pc.stride = (n + 31) / 32 * 32;
  if (n == 0) return ERI_OK;
  const size_t st = pc.stride;
  CK(pc.prim.alloc((size_t)pc.npp * 5 * st)); CK(pc.geom.alloc(7 * st)); CK(pc.aexp.alloc((size_t)pc.npp * 2 * st)); CK(pc.q.alloc(st));
  CK(pc.ao.alloc(st)); CK(pc.atom.alloc(st));
  Dev<int> sad, sbd;
  CK(sad.upload(pc.sa, g_alloc_stream)); CK(sbd.upload(pc.sb, g_alloc_stream));
  cudaStream_t as = g_alloc_stream;
  CK(cudaMemsetAsync(pc.prim.p, 0, sizeof(double) * pc.prim.n, as)); CK(cudaMemsetAsync(pc.geom.p, 0, sizeof(double) * pc.geom.n, as));
  CK(cudaMemsetAsync(pc.aexp.p, 0, sizeof(double) * pc.aexp.n, as)); CK(cudaMemsetAsync(pc.q.p, 0, sizeof(double) * st, as));
  CK(cudaMemsetAsync(pc.ao.p, 0, sizeof(int2) * st, as)); CK(cudaMemsetAsync(pc.atom.p, 0, sizeof(int2) * st, as));
  CK(launch_build_pairs(bd.sh.p, bd.pr.p, bd.xyz.p, bd.cart_off.p, sad.p, sbd.p, n, pc.Kb, pc.npp, (long)st, std::sqrt(2.0) * std::pow(PI, 1.25), pc.prim.p, pc.geom.p, pc.aexp.p,
                        pc.ao.p, pc.atom.p, as));
  CK(cudaStreamSynchronize(as));   // sad, sbd are released on return; the records can be used on any stream
  return ERI_OK;
}

// digits lost by the horizontal transfer when the 2-D integrals are built on the FIRST centre: |AB| / |PB| = p / alpha_a per quantum
double hrr_loss_of(const Basis& b, const PairClass& pc, int extra) {
  if (pc.lb + extra == 0) return 1.0;
  double ratio = 1.0;   // the power is monotonic: the largest p / alpha_a decides (one pow instead of one per primitive pair)
  for (size_t i = 0; i < pc.sa.size(); ++i) {
    const eri_shell_t& A = b.sh[pc.sa[i]]; const eri_shell_t& B = b.sh[pc.sb[i]];
    if (A.atom == B.atom) continue;   // AB = 0: the transfer adds nothing
    for (int ka = 0; ka < A.nprim; ++ka)
      for (int kb = 0; kb < B.nprim; ++kb) {
        const double ea = b.pr[A.prim_off + ka].exp, eb = b.pr[B.prim_off + kb].exp;
        ratio = std::max(ratio, (ea + eb) / ea);
      }
  }
  return std::pow(ratio, pc.lb + extra);
}

void init_pair_class(const Basis& b, int ga, int gb, PairClass& pc);

// grouped twin of a Schwarz-sorted pair set (tile family): every first shell's partner list (sorted by decreasing Q) is cut
// into HALVES of 16 slots, the halves are sorted by their head's Q and two consecutive halves make a chunk of 32 slots
// (= the lanes of a warp when the set is the ket; a bra tile is one half); padding slots have Q = -1.
constexpr int HALF = 16;
int make_grouped(const Basis& b, PairClass& pc, cudaStream_t s) {
  auto gp = std::make_unique<PairClass>();
  init_pair_class(b, pc.ga, pc.gb, *gp);
  std::map<int, std::vector<int>> by_first;
  for (int i = 0; i < pc.npair; ++i) by_first[pc.sa[i]].push_back(i);   // pc is sorted by decreasing Q, so is every group
  struct Half { double q; const std::vector<int>* idx; int begin, n; };
  std::vector<Half> halves;
  for (auto& kv : by_first)
    for (int st = 0; st < (int)kv.second.size(); st += HALF)
      halves.push_back(Half{pc.Q[kv.second[st]], &kv.second, st, std::min(HALF, (int)kv.second.size() - st)});
  std::stable_sort(halves.begin(), halves.end(), [](const Half& x, const Half& y) { return x.q > y.q; });
  const size_t nvalid = halves.size();
  if (halves.size() % 2) halves.push_back(Half{-1.0, halves.back().idx, halves.back().begin, 0});   // an all-padding half
  for (const Half& c : halves) {
    gp->half_q.push_back(c.q);
    for (int t = 0; t < HALF; ++t) {
      const int src = (*c.idx)[c.begin + (t < c.n ? t : 0)];   // padding repeats a pair of the half (valid addresses, same first shell)
      gp->sa.push_back(pc.sa[src]); gp->sb.push_back(pc.sb[src]); gp->wgt.push_back(pc.wgt[src]); gp->src.push_back(src);
      gp->Q.push_back(t < c.n ? pc.Q[src] : -1.0);
    }
  }
  gp->fill = nvalid == 0 ? 0.0 : (double)pc.npair / ((double)HALF * nvalid);
  CKI(gather_pair_class(pc, gp->src, *gp));
  pc.grouped = std::move(gp);
  return ERI_OK;
}

void init_pair_class(const Basis& b, int ga, int gb, PairClass& pc) {
  pc.ga = ga; pc.gb = gb; pc.la = b.groups[ga].l; pc.lb = b.groups[gb].l; pc.Ka = b.groups[ga].K; pc.Kb = b.groups[gb].K;
  pc.npp = pc.Ka * pc.Kb;
}

// Schwarz factors of every pair of pc (Eq. 7) through the generic store kernel on the quartets (ab|ab).
// Enqueue only: the Cartesian blocks go to a scratch buffer that all classes share (stream order keeps them apart), the
// factors to a device array of the class; schwarz_collect copies them to the host after ONE synchronisation for all classes
// (a synchronisation per class and chunk was a good part of plan creation, profiles/r02_plan.md).
struct SchwarzScratch {
  Dev<double> cart; Dev<int2> list; Dev<long long> off;
  size_t cart_cap = 0, list_cap = 0;
};
int schwarz_enqueue(PairClass& pc, Dev<double>& qdev, SchwarzScratch& sc, cudaStream_t s) {
  const int n = pc.npair;
  pc.Q.assign(n, 0.0);
  if (n == 0) return ERI_OK;
  const long nab = (long)ncart(pc.la) * ncart(pc.lb), blk = nab * nab;
  // deeply contracted sets have few pairs of many primitive quartets each ((s K=8, s K=8): some hundred pairs of 4096): one thread
  // per pair left the GPU idle for 20 ms per set (profiles/r02_plan.md); the bra primitive pairs of a pair are dealt over `split`
  // threads instead, each with its own block, and the blocks are folded before the spherical diagonal is taken
  const int split = pc.npp >= 16 ? std::min(pc.npp, 32) : 1;
  const int chunk = (int)std::max<long>(1, std::min<long>(n, (64L << 20) / (blk * split)));
  if (sc.cart_cap < (size_t)chunk * blk * split) { CK(cudaStreamSynchronize(s)); sc.cart_cap = (size_t)chunk * blk * split; CK(sc.cart.alloc(sc.cart_cap)); }
  if (sc.list_cap < (size_t)chunk * split) { CK(cudaStreamSynchronize(s)); sc.list_cap = (size_t)chunk * split; CK(sc.list.alloc(sc.list_cap)); CK(sc.off.alloc(sc.list_cap)); }
  CK(qdev.alloc(n));
  for (int start = 0; start < n; start += chunk) {
    const int m = std::min(chunk, n - start);
    CK(launch_diag_list(sc.list.p, sc.off.p, start, m, split, s));
    CK(cudaMemsetAsync(sc.cart.p, 0, sizeof(double) * (size_t)m * blk * split, s));
    Work w{}; w.bra = pc.view(); w.ket = pc.view(); w.list = sc.list.p; w.nlist = m * split; w.rys = g_rys; w.nshard = 1;
    w.kb_split = split; w.kb_items = m;
    CK(launch_generic_store(w, sc.cart.p, sc.off.p, (long)m * split, s));   // element-major blocks: coalesced accumulation
    CK(launch_fold_partials(sc.cart.p, blk, m, split, s));
    CK(launch_schwarz_diag(pc.la, pc.lb, m, (long)m * split, sc.cart.p, qdev.p + start, s));
  }
  return ERI_OK;
}
int schwarz_collect(PairClass& pc, Dev<double>& qdev) {   // after the stream has been synchronised
  if (pc.npair) CK(cudaMemcpy(pc.Q.data(), qdev.p, sizeof(double) * pc.npair, cudaMemcpyDeviceToHost));
  return ERI_OK;
}

// ---- work units -----------------------------------------------------------------------------------------------
// tile family only where at least TILE_MIN_FILL of the swept lanes has work and the bra chunks hold enough rows to amortise
// the block-end reduction (measured on cfg3)
constexpr double TILE_MIN_FILL = 0.6, TILE_MIN_BRA_FILL = 0.3, TILE_MIN_FILL_COOP = 0.25, TILE_MIN_FILL_GRAD = 0.1;
constexpr double TILE_GRAD_FILL_PP = 0.65, TILE_GRAD_FILL_PP_SHORT = 0.35;   // tile gradient kernel against the primitive-parallel one: lane fill below which the latter
                                                                             // takes the unit, for 8 or more / fewer primitive quartets per quartet (measured on cfg4)
constexpr long long PGRAD_MIN_NPP = 3;    // primitive quartets per quartet from which the primitive-parallel gradient kernel fills its lanes (it packs 32 / npp quartets into a warp)
constexpr long long COOP_GRAD_MIN_TASKS = 32768;   // some twenty waves of 12 warps on 148 SMs: the tail of a unit is a wave of heavy tasks
constexpr double HRR_LOSS_MAX_GRAD = 1.0e5;   // gradient tolerance is 1e-8 Ha/Bohr absolute
constexpr double HRR_LOSS_MAX = 1.0e3;   // at most three digits (tile family; otherwise the cooperative family chooses the centre)

struct Unit {
  int P = 0, R = 0; bool same = false;
  int BI = GENERIC_BI, BJ = GENERIC_BJ, nrows = 0, nblocks = 0;
  int gBI = GENERIC_GRAD_BI, gBJ = GENERIC_GRAD_BJ, g_nrows = 0, g_nblocks = 0;
  int kernel = 0, kernel_grad = 0;
  long long quartets = 0;
  double flops = 0, flops_grad = 0;
  float last_ms = 0, last_ms_grad = 0;
  std::vector<int> h_count;
  int index = 0;                            // position in eri_plan::units
  Dev<int> ket_count, row_off, g_row_off;
  Dev<int> ket_count_dyn;                   // density-weighted call: kept prefix per bra pair under tau / P_{ab|cd}
  Dev<int> t_row_slot, t_row_off; int t_nrows = 0, t_nblocks = 0, tBI = 0; long long t_slots = 0;   // tile family
  Dev<int2> list; int nlist = 0;            // list mode
  Dev<long long> coff;                      // list mode, store kernel
};

}  // namespace
}  // namespace eri

using namespace eri;

struct eri_plan {
  Basis basis;
  bool is_list = false, want_grad = false;
  double thr = 0.0;
  int kernel_mode = 0, timing = 0, shard = 0, nshard = 1, serial = 0;
  double tile_fill_scale = 1.0;                       // eri_plan_set_tuning: multiplies the tile family's fill thresholds
  long long grad_min_tasks = COOP_GRAD_MIN_TASKS;     // eri_plan_set_tuning: tasks per unit below which the cooperative gradient run is halved
  long long pgrad_min_npp = PGRAD_MIN_NPP;            // eri_plan_set_tuning: primitive quartets per quartet from which the primitive-parallel gradient kernel serves a unit
  std::vector<std::unique_ptr<PairClass>> pcs;
  std::vector<std::unique_ptr<Unit>> units;
  Dev<int> sh_l, sh_sph, sh_cart, sph2sh, cart2sh;
  Dev<double> Dc, Jc, Kc, Dh, Jh, Kh, gJd, gKd;   // Cartesian workspaces; device staging for the *_host entry points
  // density-weighted screening (eri_plan_build_jk_dscreen): AO -> shell group, group sub-block maxima of |D|, per unit the
  // effective threshold and the number of quartets that passed in the last call
  Dev<int> ao_group; Dev<unsigned long long> pmax, ds_kept; Dev<double> thr_eff; Dev<DscreenUnit> ds_units;
  int ds_max_nbra = 0; bool ds_ready = false, ds_active = false;
  ShellMap map{};
  eri_stats_t stats{};
  std::vector<cudaEvent_t> ev;   // timing mode: ev[k] before unit k, ev[n] after the last one (no host sync in between)
  bool ev_pending = false, ev_grad = false;
  // concurrent mode (default outside timing mode): the units are independent (they merge by atomic add), so they
  // are dealt over a small pool of streams, heaviest first, forked from and joined to the caller's stream with events
  std::vector<cudaStream_t> pool; std::vector<cudaEvent_t> pool_ev; cudaEvent_t fork_ev = nullptr;
  std::vector<int> order, order_grad;   // unit indices by decreasing cost
  // CUDA graph of the concurrent J/K launch schedule (the class kernels touch plan-owned buffers only): [0] plain, [1] density-weighted
  // call.  Captured at the second call of a selection (the first one sets the kernels' attributes), replayed afterwards: one
  // graph launch instead of some hundred kernel launches and stream/event calls -- the small workloads are launch-bound.
  cudaGraphExec_t jk_graph[2] = {nullptr, nullptr};
  int jk_graph_gen[2] = {-1, -1}, jk_calls[2] = {0, 0}, sel_gen = 0;
  bool graphs_ok = true;
  ~eri_plan() {
    for (cudaGraphExec_t g : jk_graph) if (g) cudaGraphExecDestroy(g);
    for (cudaEvent_t e : ev) cudaEventDestroy(e);
    for (cudaEvent_t e : pool_ev) cudaEventDestroy(e);
    for (cudaStream_t st : pool) cudaStreamDestroy(st);
    if (fork_ev) cudaEventDestroy(fork_ev);
  }
};

namespace eri {
namespace {

int make_shell_map(eri_plan& pl, cudaStream_t s) {
  const Basis& b = pl.basis;
  const int ns = (int)b.sh.size();
  std::vector<int> l(ns), so(ns), co(ns), s2s(b.nao), c2s(b.nao_cart);
  for (int i = 0; i < ns; ++i) {
    l[i] = b.sh[i].l; so[i] = b.sh[i].ao_off; co[i] = b.cart_off[i];
    for (int k = 0; k < nsph(l[i]); ++k) s2s[so[i] + k] = i;
    for (int k = 0; k < ncart(l[i]); ++k) c2s[co[i] + k] = i;
  }
  CK(pl.sh_l.upload(l, s)); CK(pl.sh_sph.upload(so, s)); CK(pl.sh_cart.upload(co, s));
  CK(pl.sph2sh.upload(s2s, s)); CK(pl.cart2sh.upload(c2s, s));
  CK(cudaStreamSynchronize(s));
  pl.map = ShellMap{pl.sh_l.p, pl.sh_sph.p, pl.sh_cart.p, pl.sph2sh.p, pl.cart2sh.p, ns, b.nao, b.nao_cart};
  const size_t n2 = (size_t)b.nao_cart * b.nao_cart;
  CK(pl.Dc.alloc(n2)); CK(pl.Jc.alloc(n2)); CK(pl.Kc.alloc(n2));
  return ERI_OK;
}

double canonical_flops(int la, int lb, int lc, int ld, int ka, int kb, int kc, int kd, int deriv) {
  // DESIGN.md "FLOP model" (FMA = 2): the work the Rys method has to do, independent of kernel organisation.
  const int L = la + lb + lc + ld + (deriv ? 1 : 0), N = L / 2 + 1;
  const int nmax = la + lb + (deriv ? 1 : 0), mmax = lc + ld + (deriv ? 1 : 0);
  const double fvrr = 6.0 * (nmax + 1) * (mmax + 1);
  double fh = 0.0;
  for (int j = 1; j <= lb; ++j) fh += (double)(nmax - j + 1) * (mmax + 1);
  for (int l = 1; l <= ld; ++l) fh += (double)(mmax - l + 1) * (la + 1) * (lb + 1);
  const double fhrr = 2.0 * fh;
  const double nc = (double)ncart(la) * ncart(lb) * ncart(lc) * ncart(ld);
  const double kprod = (double)ka * kb * kc * kd;
  if (!deriv) {
    const double fprim = 60.0 + 56.0 * N + N * (25.0 + 3.0 * (fvrr + fhrr)) + 3.0 * N * nc;
    const double nsa = nsph(la), nsb = nsph(lb), nsc = nsph(lc), nsd = nsph(ld);
    const double nca = ncart(la), ncb = ncart(lb), ncc = ncart(lc), ncd = ncart(ld);
    const double fc2s = 2.0 * (nsa * nca * ncb * ncc * ncd + nsa * nsb * ncb * ncc * ncd + nsa * nsb * nsc * ncc * ncd + nsa * nsb * nsc * nsd * ncd);
    return kprod * fprim + fc2s + 12.0 * nsa * nsb * nsc * nsd;
  }
  // gradient: per root and element 3 pair products + 9 derivative FMAs; 18 density FMAs per element and primitive quartet
  const double fprim = 60.0 + 56.0 * N + N * (25.0 + 3.0 * (fvrr + fhrr)) + 21.0 * N * nc + 36.0 * nc;
  return kprod * fprim;
}

// dense-mode decomposition of one unit for a (BI, BJ) tile shape
void make_rows(const std::vector<int>& count, int BI, int BJ, std::vector<int>& row_off) {
  const int nb = (int)count.size(), nrows = (nb + BI - 1) / BI;
  row_off.assign(nrows + 1, 0);
  for (int r = 0; r < nrows; ++r) {
    int mx = 0;
    for (int i = r * BI; i < std::min(nb, (r + 1) * BI); ++i) mx = std::max(mx, count[i]);
    row_off[r + 1] = row_off[r] + (mx + BJ - 1) / BJ;
  }
}

int select_kernels(eri_plan& pl, Unit& u, cudaStream_t s) {
  const PairClass& P = *pl.pcs[u.P]; const PairClass& R = *pl.pcs[u.R];
  TunedInfo ti{};
  u.kernel = 0; u.BI = GENERIC_BI; u.BJ = GENERIC_BJ;
  const bool canonical = P.la >= P.lb && R.la >= R.lb && (P.la > R.la || (P.la == R.la && P.lb >= R.lb));
  if (pl.kernel_mode != 1 && canonical && tuned_jk_info(P.la, P.lb, R.la, R.lb, P.npp, R.npp, &ti)) {
    // the register family (kind 1) builds the 2-D integrals on the first centre of each pair like the tile family: same guard
    // (the cooperative family chooses the centre per primitive pair; the generic kernel does too)
    if (ti.kind != 1 || (P.hrr_loss <= HRR_LOSS_MAX && R.hrr_loss <= HRR_LOSS_MAX)) { u.kernel = ti.kind; u.BI = ti.BI; u.BJ = ti.BJ; }
  }
  // tile family: dense mode, and only where building the 2-D integrals on the first centre of every pair is safe
  u.kernel_grad = 0; u.gBI = GENERIC_GRAD_BI; u.gBJ = GENERIC_GRAD_BJ;
  if (pl.kernel_mode == 0 && canonical && !pl.is_list && P.grouped && R.grouped) {
    const PairClass& gb = *P.grouped; const PairClass& gk = *R.grouped;
    if (u.t_nblocks == 0) {   // blocks of the tile decomposition (independent of the class kernel): once per unit
      const int nbh = (int)gb.half_q.size(), nkc = (int)gk.half_q.size() / 2;
      std::vector<int> slot, off{0};
      long long slots = 0;
      for (int hb = 0; hb < nbh; ++hb) {   // one block per (bra half, ket chunk of the prefix that passes Schwarz)
        const double qb = gb.half_q[hb];
        if (qb < 0.0) continue;
        int lo = 0, hi = nkc;   // the first half of a ket chunk carries the chunk's largest factor
        if (pl.thr > 0.0) { while (lo < hi) { const int mid = (lo + hi) / 2; if (qb * gk.half_q[2 * mid] >= pl.thr) lo = mid + 1; else hi = mid; } }
        else lo = nkc;
        if (u.same) lo = std::min(lo, hb / 2 + 1);
        if (lo == 0) continue;
        slot.push_back(HALF * hb); off.push_back(off.back() + lo);
        // lane slots actually swept = rows with work x 32 (the kernel skips the other rows; rows are sorted within the half)
        // rows of the half and ket chunks are both sorted by decreasing factor: the number of rows with work can only
        // shrink from one chunk to the next (two-pointer sweep instead of a scan of the 16 rows per chunk)
        int nr = 0;
        while (nr < HALF && gb.Q[HALF * hb + nr] >= 0.0) ++nr;
        for (int ck = 0; ck < lo; ++ck) {
          while (nr > 0 && gb.Q[HALF * hb + nr - 1] * gk.half_q[2 * ck] < pl.thr) --nr;
          slots += 32 * nr;
        }
      }
      u.t_slots = slots; u.t_nrows = (int)slot.size(); u.t_nblocks = off.back();
      CK(u.t_row_slot.upload(slot, s)); CK(u.t_row_off.upload(off, s));
    }
    const double fill = u.t_slots > 0 ? (double)u.quartets / (double)u.t_slots : 0.0;
    if (P.hrr_loss <= HRR_LOSS_MAX && R.hrr_loss <= HRR_LOSS_MAX && tile_jk_info(P.la, P.lb, R.la, R.lb, &ti)) {
      // the register family (kind 1) is hard to beat on sparsely filled tiles; the cooperative family (kind 2) is not
      const double fs = pl.tile_fill_scale;
      const bool take = u.kernel == 1 ? (fill >= fs * TILE_MIN_FILL && gb.fill >= fs * TILE_MIN_BRA_FILL) : fill >= fs * (ti.TQ >= 5 ? TILE_MIN_FILL : TILE_MIN_FILL_COOP);
      if (take) { u.kernel = 3; u.tBI = ti.BI; }
    }
    // gradient: one more quantum is transferred (lb + 1, ld + 1 is not raised), so the loss bound is one power higher
    if (pl.want_grad && fill >= pl.tile_fill_scale * TILE_MIN_FILL_GRAD && P.hrr_loss_grad <= HRR_LOSS_MAX_GRAD && R.hrr_loss <= HRR_LOSS_MAX_GRAD &&
        tuned_grad_info(P.la, P.lb, R.la, R.lb, P.npp, R.npp, &ti)) {
      // deeply contracted units on badly filled tiles (a contracted second ket shell has few partners per first shell: half the
      // lanes idle, profiles/r02_cfg4.md) are left to the primitive-parallel kernel below, whose lanes own primitive quartets
      TunedInfo tp{};
      const long long npq = (long long)P.npp * R.npp;
      // (the classes of 54 Cartesian elements run the axis-team variant of the tile kernel, three threads and two barriers per
      // quartet: there the primitive-parallel kernel wins or ties at any fill once a quartet has three primitive quartets)
      const int ne = ncart(P.la) * ncart(P.lb) * ncart(R.la) * ncart(R.lb);
      const bool pp_better = (ne >= 54 || fill < pl.tile_fill_scale * (npq >= 8 ? TILE_GRAD_FILL_PP : TILE_GRAD_FILL_PP_SHORT)) && npq >= pl.pgrad_min_npp &&
                             pp_grad_info(P.la, P.lb, R.la, R.lb, &tp);
      if (!pp_better) { u.kernel_grad = 3; u.gBI = ti.BI; }
    }
  }
  // cooperative gradient kernel for what the tile gradient kernel does not serve (it chooses the build centre itself)
  if (pl.kernel_mode != 1 && pl.want_grad && canonical && !pl.is_list && u.kernel_grad == 0 && coop_grad_info(P.la, P.lb, R.la, R.lb, &ti)) {
    u.kernel_grad = 2; u.gBI = ti.BI; u.gBJ = ti.BJ;
    // a warp walks its task's bra pairs one after the other: units of few, heavy quartets (the contracted core shells,
    // K^4 = 4096 primitive quartets each) get shorter runs so that they still spread over the SMs
    // deeply contracted units of the low-l classes: the lanes of the warp own primitive quartets (pp_grad.cuh); the 2-D integrals are
    // built on the first centres there, so the same guard as for the tile gradient kernel applies
    if ((long long)P.npp * R.npp >= pl.pgrad_min_npp && P.hrr_loss_grad <= HRR_LOSS_MAX_GRAD && R.hrr_loss <= HRR_LOSS_MAX_GRAD &&
        pp_grad_info(P.la, P.lb, R.la, R.lb, &ti)) { u.kernel_grad = 4; u.gBI = ti.BI; u.gBJ = ti.BJ; }
    // (the primitive-parallel kernel packs 32 / npp bra pairs of a run into one warp: its runs stay at least that long)
    const long long npq = (long long)P.npp * R.npp;
    const int min_run = u.kernel_grad == 4 && npq < 32 ? (int)std::min<long long>(16, 32 / npq) : 1;
    while (u.gBI > min_run && u.gBI / 2 >= min_run && u.quartets / u.gBI < pl.grad_min_tasks) u.gBI /= 2;
  }
  if (!pl.is_list) {
    std::vector<int> ro;
    make_rows(u.h_count, u.BI, u.BJ, ro);
    u.nrows = (int)ro.size() - 1; u.nblocks = ro.back();
    CK(u.row_off.upload(ro, s));
    if (pl.want_grad) {
      make_rows(u.h_count, u.gBI, u.gBJ, ro);
      u.g_nrows = (int)ro.size() - 1; u.g_nblocks = ro.back();
      CK(u.g_row_off.upload(ro, s));
    }
    CK(cudaStreamSynchronize(s));
  }
  return ERI_OK;
}

Work make_work(const eri_plan& pl, const Unit& u, bool grad) {
  Work w{};
  w.bra = pl.pcs[u.P]->view(); w.ket = pl.pcs[u.R]->view();
  w.ket_count = u.ket_count.p;
  if (pl.ds_active && !grad) { w.ket_count = u.ket_count_dyn.p; w.thr_dev = pl.thr_eff.p + u.index; }
  w.row_off = grad ? u.g_row_off.p : u.row_off.p;
  w.nrows = grad ? u.g_nrows : u.nrows;
  w.thr = pl.thr;
  w.grad_ch = u.gBI;
  if (grad ? u.kernel_grad == 3 : u.kernel == 3) {
    w.bra = pl.pcs[u.P]->grouped->view(); w.ket = pl.pcs[u.R]->grouped->view();
    w.row_off = u.t_row_off.p; w.row_slot = u.t_row_slot.p; w.nrows = u.t_nrows;
  }
  w.same = u.same ? 1 : 0;
  w.list = pl.is_list ? u.list.p : nullptr; w.nlist = u.nlist;
  w.rys = g_rys; w.D = pl.Dc.p; w.J = pl.Jc.p; w.K = pl.Kc.p; w.nao = pl.basis.nao_cart;
  w.shard = pl.shard; w.nshard = pl.nshard;
  return w;
}

constexpr int POOL_STREAMS = 8;
constexpr long long POOL_BIG_BLOCKS = 4 * 148;   // at least four blocks per SM: the launch fills the GPU

// which tuned instantiations this process has launched (eri_kernel_launched; read by the test-suite's coverage check)
std::mutex g_log_mu;
std::set<std::string> g_launched;
void log_launch(const char* fam, const Work& w) {
  char buf[64]; snprintf(buf, sizeof buf, "%s %d %d %d %d", fam, w.bra.la, w.bra.lb, w.ket.la, w.ket.lb);
  std::lock_guard<std::mutex> lk(g_log_mu);
  g_launched.insert(buf);
}

int launch_unit(eri_plan& pl, Unit& u, bool grad, double* gJ, double* gK, cudaStream_t s) {
  Work w = make_work(pl, u, grad);
  w.gJ = gJ; w.gK = gK;
  {
    const int k = grad ? u.kernel_grad : u.kernel;
    TunedInfo ti{};
    const char* fam = grad ? (k == 3 ? "tgrad" : k == 2 ? "cgrad" : k == 4 ? "pgrad" : "generic_grad")
                           : (k == 3 ? "tile" : k == 2 ? "coop" : k == 1 ? "reg" : "generic");
    (void)ti;
    log_launch(fam, w);
  }
  if (!grad) {
    if (u.kernel == 0) CK(launch_generic_jk(w, u.nblocks, s));
    else if (u.kernel == 3) CK(launch_tile_jk_class(w, u.t_nblocks, s));
    else CK(launch_tuned_jk(w, u.nblocks, s));
  } else {
    if (u.kernel_grad == 0) CK(launch_generic_grad(w, u.g_nblocks, s));
    else if (u.kernel_grad == 2) CK(launch_coop_grad_class(w, u.g_nblocks, s));
    else if (u.kernel_grad == 4) CK(launch_pp_grad_class(w, u.g_nblocks, s));
    else CK(launch_tuned_grad(w, u.t_nblocks, s));
  }
  return ERI_OK;
}

int ensure_pool(eri_plan& pl) {
  if (!pl.pool.empty()) return ERI_OK;
  CK(cudaEventCreateWithFlags(&pl.fork_ev, cudaEventDisableTiming));
  for (int k = 0; k < POOL_STREAMS; ++k) {
    cudaStream_t st; CK(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking)); pl.pool.push_back(st);
    cudaEvent_t e; CK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming)); pl.pool_ev.push_back(e);
  }
  return ERI_OK;
}

// the concurrent launch schedule: units by decreasing cost, the large ones on the caller's stream, the small ones on the pool
int run_units_concurrent(eri_plan& pl, bool grad, double* gJ, double* gK, cudaStream_t s) {
  const int nu = (int)pl.units.size();
  std::vector<int>& order = grad ? pl.order_grad : pl.order;
  if ((int)order.size() != nu) {
    order.resize(nu);
    for (int k = 0; k < nu; ++k) order[k] = k;
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) {
      return (grad ? pl.units[x]->flops_grad : pl.units[x]->flops) > (grad ? pl.units[y]->flops_grad : pl.units[y]->flops); });
  }
  CK(cudaEventRecord(pl.fork_ev, s));
  for (cudaStream_t st : pl.pool) CK(cudaStreamWaitEvent(st, pl.fork_ev, 0));
  // launches that fill the GPU by themselves stay on the caller's stream, one after the other (they only disturb each other
  // when they overlap); the many small ones (deeply contracted pair sets with few pairs) share the pool and fill the gaps
  int small = 0;
  for (int k = 0; k < nu; ++k) {
    Unit& u = *pl.units[order[k]];
    const long long blocks = grad ? (u.kernel_grad == 3 ? u.t_nblocks : u.g_nblocks) : (u.kernel == 3 ? u.t_nblocks : u.nblocks);
    const bool big = blocks / pl.nshard >= POOL_BIG_BLOCKS;
    CKI(launch_unit(pl, u, grad, gJ, gK, big ? s : pl.pool[small++ % POOL_STREAMS]));
  }
  for (int k = 0; k < POOL_STREAMS; ++k) { CK(cudaEventRecord(pl.pool_ev[k], pl.pool[k])); CK(cudaStreamWaitEvent(s, pl.pool_ev[k], 0)); }
  return ERI_OK;
}

int run_units(eri_plan& pl, bool grad, double* gJ, double* gK, cudaStream_t s) {
  const int nu = (int)pl.units.size();
  if (pl.timing) {   // serial, one event between launches: per-unit device times
    while ((int)pl.ev.size() < nu + 1) { cudaEvent_t e; CK(cudaEventCreate(&e)); pl.ev.push_back(e); }
    for (int k = 0; k < nu; ++k) {
      CK(cudaEventRecord(pl.ev[k], s));
      CKI(launch_unit(pl, *pl.units[k], grad, gJ, gK, s));
    }
    CK(cudaEventRecord(pl.ev[nu], s)); pl.ev_pending = true; pl.ev_grad = grad;
    return ERI_OK;
  }
  if (nu < 2 || pl.serial) {
    for (int k = 0; k < nu; ++k) CKI(launch_unit(pl, *pl.units[k], grad, gJ, gK, s));
    return ERI_OK;
  }
  CKI(ensure_pool(pl));
  if (!grad && pl.graphs_ok) {
    const int gi = pl.ds_active ? 1 : 0;
    if (pl.jk_graph[gi] && pl.jk_graph_gen[gi] == pl.sel_gen) { CK(cudaGraphLaunch(pl.jk_graph[gi], s)); return ERI_OK; }
    if (pl.jk_graph_gen[gi] != pl.sel_gen) { pl.jk_graph_gen[gi] = pl.sel_gen; pl.jk_calls[gi] = 0; if (pl.jk_graph[gi]) { cudaGraphExecDestroy(pl.jk_graph[gi]); pl.jk_graph[gi] = nullptr; } }
    if (pl.jk_calls[gi]++ >= 1) {   // second call of this selection: capture the schedule, then replay it
      cudaGraph_t g = nullptr;
      if (cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
        const int rc = run_units_concurrent(pl, false, nullptr, nullptr, s);
        const cudaError_t ec = cudaStreamEndCapture(s, &g);
        if (rc == ERI_OK && ec == cudaSuccess && g && cudaGraphInstantiate(&pl.jk_graph[gi], g, 0) == cudaSuccess) {
          cudaGraphDestroy(g);
          CK(cudaGraphLaunch(pl.jk_graph[gi], s));
          return ERI_OK;
        }
        if (g) cudaGraphDestroy(g);
        pl.jk_graph[gi] = nullptr;
      }
      cudaGetLastError();        // capture is an optimisation: on any failure fall back to plain launches for good
      pl.graphs_ok = false;
    }
  }
  return run_units_concurrent(pl, grad, gJ, gK, s);
}

int plan_common(eri_plan& pl, const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim,
                const double* coords, int natm, cudaStream_t s) {
  CKI(make_basis(shells, nshell, prims, nprim, coords, natm, pl.basis));   // argument errors first: they need no device
  CKI(ensure_init());
  CKI(make_shell_map(pl, s));
  return ERI_OK;
}

int create_dense_plan(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim, const double* coords, int natm,
                      double thr, int want_grad, cudaStream_t s, eri_plan& pl) {
  const auto t0 = std::chrono::steady_clock::now();
  if (!(thr >= 0.0)) return fail(ERI_ERR_BAD_ARG, "schwarz_thr must be >= 0");
  CKI(plan_common(pl, shells, nshell, prims, nprim, coords, natm, s));
  pl.thr = thr; pl.want_grad = want_grad != 0;
  const Basis& b = pl.basis;
  const int ng = (int)b.groups.size();
  auto lap = [&, last = t0]() mutable { const auto now = std::chrono::steady_clock::now(); const double ms = std::chrono::duration<double, std::milli>(now - last).count(); last = now; return ms; };
  pl.stats.plan_ms_init = lap();
  // pair sets |ab, KaKb} for group(a) >= group(b) (groups sorted by (l,K), so la >= lb) -- Alg. 1 lines 3-6
  std::vector<std::unique_ptr<PairClass>> all;
  std::deque<Dev<double>> qdev;   // Schwarz factors of the classes on the device until the one synchronisation below
  // the Schwarz passes of the pair sets are independent: dealt over the plan's stream pool (each stream its own scratch), so that
  // the sets with few, heavy pairs (the K = 8 core shells, the f shells) overlap instead of running one after the other
  CKI(ensure_pool(pl));
  constexpr int NSCR = 4;
  SchwarzScratch scratch[NSCR];
  BasisDev bdev;
  CKI(upload_basis(b, bdev, s));
  CK(cudaStreamSynchronize(s));   // the pool streams are not ordered behind the caller's stream: everything queued there is done first
  double qmax = 0.0;
  long long pairs_total = 0;
  for (int ga = 0; ga < ng; ++ga)
    for (int gb = 0; gb <= ga; ++gb) {
      auto pc = std::make_unique<PairClass>();
      init_pair_class(b, ga, gb, *pc);
      const auto& A = b.groups[ga].shells; const auto& B = b.groups[gb].shells;
      for (size_t ia = 0; ia < A.size(); ++ia)
        for (size_t ib = 0; ib < (ga == gb ? ia + 1 : B.size()); ++ib) {
          pc->sa.push_back(A[ia]); pc->sb.push_back(B[ib]); pc->wgt.push_back(A[ia] == B[ib] ? 0.5 : 1.0);
        }
      pairs_total += (long long)pc->sa.size();
      CKI(build_pair_class_device(bdev, *pc));
      qdev.emplace_back();
      CKI(schwarz_enqueue(*pc, qdev.back(), scratch[all.size() % NSCR], pl.pool[all.size() % NSCR]));
      all.push_back(std::move(pc));
    }
  for (int k = 0; k < NSCR; ++k) CK(cudaStreamSynchronize(pl.pool[k]));
  for (size_t k = 0; k < all.size(); ++k) {
    CKI(schwarz_collect(*all[k], qdev[k]));
    for (double q : all[k]->Q) qmax = std::max(qmax, q);
  }
  qdev.clear();
  pl.stats.plan_ms_schwarz = lap();
  // prescreen (Alg. 1 line 7), sort by decreasing bound (the paper bins, Eq. 6; sorting is the limit of fine bins)
  long long pairs_kept = 0;
  for (auto& pc : all) {
    std::vector<int> idx;
    for (int i = 0; i < pc->npair; ++i) if (thr == 0.0 || pc->Q[i] * qmax >= thr) idx.push_back(i);
    std::stable_sort(idx.begin(), idx.end(), [&](int x, int y) { return pc->Q[x] > pc->Q[y]; });
    if (idx.empty()) continue;
    auto np = std::make_unique<PairClass>();
    init_pair_class(b, pc->ga, pc->gb, *np);
    for (int i : idx) { np->sa.push_back(pc->sa[i]); np->sb.push_back(pc->sb[i]); np->wgt.push_back(pc->wgt[i]); np->Q.push_back(pc->Q[i]); }
    CKI(gather_pair_class(*pc, idx, *np));
    np->hrr_loss = hrr_loss_of(b, *np, 0); np->hrr_loss_grad = hrr_loss_of(b, *np, 1);
    CKI(make_grouped(b, *np, s));
    pairs_kept += np->npair;
    pl.pcs.push_back(std::move(np));
  }
  all.clear();
  // canonical order of pair sets: by (la, lb), then groups; bra set >= ket set gives (la,lb) >= (lc,ld)
  std::sort(pl.pcs.begin(), pl.pcs.end(), [](const std::unique_ptr<PairClass>& x, const std::unique_ptr<PairClass>& y) {
    return std::make_tuple(x->la, x->lb, x->ga, x->gb) < std::make_tuple(y->la, y->lb, y->ga, y->gb);
  });
  pl.stats.plan_ms_pairs = lap();
  // work units: bra set P >= ket set R; per bra pair the kept kets are a prefix of the sorted ket set (reading R7)
  long long qkept = 0; double flops = 0, flops_g = 0;
  std::vector<std::pair<int, int>> cand;
  for (int P = 0; P < (int)pl.pcs.size(); ++P) for (int R = 0; R <= P; ++R) cand.push_back({P, R});
  std::vector<std::unique_ptr<Unit>> built(cand.size());
  CKI(parallel_ranges((int)cand.size(), 8, [&](int lo_u, int hi_u) {
    for (int c = lo_u; c < hi_u; ++c) {
      const int P = cand[c].first, R = cand[c].second;
      const PairClass& bp = *pl.pcs[P]; const PairClass& kp = *pl.pcs[R];
      auto u = std::make_unique<Unit>();
      u->P = P; u->R = R; u->same = (P == R);
      u->h_count.resize(bp.npair);
      long long tot = 0;
      for (int i = 0; i < bp.npair; ++i) {
        int cnt = kp.npair;
        if (thr > 0.0) {   // largest prefix with Q_i * Q_j >= thr
          int lo = 0, hi = kp.npair;
          while (lo < hi) { const int mid = (lo + hi) / 2; if (bp.Q[i] * kp.Q[mid] >= thr) lo = mid + 1; else hi = mid; }
          cnt = lo;
        }
        if (u->same) cnt = std::min(cnt, i + 1);
        u->h_count[i] = cnt; tot += cnt;
      }
      if (tot == 0) continue;
      u->quartets = tot;
      u->flops = tot * canonical_flops(bp.la, bp.lb, kp.la, kp.lb, bp.Ka, bp.Kb, kp.Ka, kp.Kb, 0);
      u->flops_grad = tot * canonical_flops(bp.la, bp.lb, kp.la, kp.lb, bp.Ka, bp.Kb, kp.Ka, kp.Kb, 1);
      CK(u->ket_count.upload(u->h_count, s));
      CKI(select_kernels(pl, *u, s));
      built[c] = std::move(u);
    }
    return (int)ERI_OK;
  }));
  for (auto& u : built) {
    if (!u) continue;
    qkept += u->quartets; flops += u->flops; flops_g += u->flops_grad;
    u->index = (int)pl.units.size();
    pl.units.push_back(std::move(u));
  }
  CK(cudaStreamSynchronize(s));
  pl.stats.plan_ms_units = lap();
  eri_stats_t& st = pl.stats;
  st.nshell = nshell; st.nao = b.nao; st.nao_cart = b.nao_cart; st.natm = natm;
  st.n_shell_groups = ng; st.n_pair_classes = (int)pl.pcs.size(); st.n_quartet_classes = (int)pl.units.size();
  st.launches_per_call = (int)pl.units.size() + 5;
  st.pairs_total = pairs_total; st.pairs_kept = pairs_kept;
  st.quartets_total = pairs_total * (pairs_total + 1) / 2; st.quartets_kept = qkept;
  st.canonical_flops = flops; st.canonical_flops_grad = flops_g;
  st.plan_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  return ERI_OK;
}

// list plan: pair sets from the distinct ordered shell pairs of the list, in the order given (any l order)
int create_list_plan(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim, const double* coords, int natm,
                     const int32_t* quartets, int n, cudaStream_t s, eri_plan& pl, std::vector<long long>* cart_off_out,
                     long long* cart_total) {
  const auto t0 = std::chrono::steady_clock::now();
  if (n < 0 || (n > 0 && !quartets)) return fail(ERI_ERR_BAD_ARG, "bad quartet list");
  CKI(plan_common(pl, shells, nshell, prims, nprim, coords, natm, s));
  pl.is_list = true;
  const Basis& b = pl.basis;
  for (int t = 0; t < 4 * n; ++t) if (quartets[t] < 0 || quartets[t] >= nshell) return fail(ERI_ERR_BAD_ARG, "quartet %d names shell %d", t / 4, quartets[t]);
  std::map<std::pair<int, int>, int> class_of;            // (group, group) -> pair set index
  std::vector<std::map<std::pair<int, int>, int>> pair_of;  // per pair set: (shell, shell) -> pair index
  auto pair_id = [&](int i, int j, int& cls) {
    const std::pair<int, int> key{b.group_of[i], b.group_of[j]};
    auto it = class_of.find(key);
    if (it == class_of.end()) {
      it = class_of.emplace(key, (int)pl.pcs.size()).first;
      auto pc = std::make_unique<PairClass>(); init_pair_class(b, key.first, key.second, *pc);
      pl.pcs.push_back(std::move(pc)); pair_of.emplace_back();
    }
    cls = it->second;
    auto& pm = pair_of[cls];
    auto jt = pm.find({i, j});
    if (jt == pm.end()) { jt = pm.emplace(std::make_pair(i, j), (int)pl.pcs[cls]->sa.size()).first; pl.pcs[cls]->sa.push_back(i); pl.pcs[cls]->sb.push_back(j); }
    return jt->second;
  };
  std::map<std::pair<int, int>, int> unit_of;
  std::vector<std::vector<int2>> lists; std::vector<std::vector<long long>> coffs;
  long long ctot = 0;
  if (cart_off_out) cart_off_out->resize(n);
  double flops = 0;
  for (int t = 0; t < n; ++t) {
    int cb, ck;
    const int pb = pair_id(quartets[4 * t], quartets[4 * t + 1], cb), pk = pair_id(quartets[4 * t + 2], quartets[4 * t + 3], ck);
    auto it = unit_of.find({cb, ck});
    if (it == unit_of.end()) {
      it = unit_of.emplace(std::make_pair(cb, ck), (int)pl.units.size()).first;
      auto u = std::make_unique<Unit>(); u->P = cb; u->R = ck; pl.units.push_back(std::move(u)); lists.emplace_back(); coffs.emplace_back();
    }
    lists[it->second].push_back(make_int2(pb, pk));
    coffs[it->second].push_back(ctot);
    if (cart_off_out) (*cart_off_out)[t] = ctot;
    long long blk = 1; for (int x = 0; x < 4; ++x) blk *= ncart(b.sh[quartets[4 * t + x]].l);
    ctot += blk;
  }
  if (cart_total) *cart_total = ctot;
  for (auto& pc : pl.pcs) { CKI(upload_pair_class(b, *pc, s)); pc->hrr_loss = hrr_loss_of(b, *pc, 0); pc->hrr_loss_grad = hrr_loss_of(b, *pc, 1); }
  for (size_t k = 0; k < pl.units.size(); ++k) {
    Unit& u = *pl.units[k];
    u.nlist = (int)lists[k].size(); u.quartets = u.nlist;
    const PairClass& bp = *pl.pcs[u.P]; const PairClass& kp = *pl.pcs[u.R];
    u.flops = u.quartets * canonical_flops(bp.la, bp.lb, kp.la, kp.lb, bp.Ka, bp.Kb, kp.Ka, kp.Kb, 0);
    flops += u.flops;
    CK(u.list.upload(lists[k], s));
    if (cart_off_out) CK(u.coff.upload(coffs[k], s));
    CKI(select_kernels(pl, u, s));
  }
  CK(cudaStreamSynchronize(s));
  eri_stats_t& st = pl.stats;
  st.nshell = nshell; st.nao = b.nao; st.nao_cart = b.nao_cart; st.natm = natm;
  st.n_shell_groups = (int)b.groups.size(); st.n_pair_classes = (int)pl.pcs.size(); st.n_quartet_classes = (int)pl.units.size();
  st.launches_per_call = (int)pl.units.size() + 5;
  st.quartets_total = n; st.quartets_kept = n; st.canonical_flops = flops;
  for (auto& pc : pl.pcs) { st.pairs_total += pc->npair; st.pairs_kept += pc->npair; }
  st.plan_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  return ERI_OK;
}

int build_jk(eri_plan& pl, const double* D, double* J, double* K, cudaStream_t s) {
  if (!D || !J || !K) return fail(ERI_ERR_BAD_ARG, "null matrix pointer");
  CKI(ensure_init());   // device check
  const size_t n2 = (size_t)pl.basis.nao_cart * pl.basis.nao_cart;
  if (pl.basis.nao == 0) return ERI_OK;
  CK(launch_sph2cart(pl.map, D, pl.Dc.p, s));
  CK(cudaMemsetAsync(pl.Jc.p, 0, n2 * sizeof(double), s));
  CK(cudaMemsetAsync(pl.Kc.p, 0, n2 * sizeof(double), s));
  CKI(run_units(pl, false, nullptr, nullptr, s));
  if (pl.is_list) {
    CK(launch_cart2sph(pl.map, pl.Jc.p, J, 1.0, 0, s));
    CK(launch_cart2sph(pl.map, pl.Kc.p, K, 1.0, 0, s));
  } else {   // reading R9: J = 2 (Jt + Jt^T), K = Kt + Kt^T
    CK(launch_cart2sph(pl.map, pl.Jc.p, J, 2.0, 1, s));
    CK(launch_cart2sph(pl.map, pl.Kc.p, K, 1.0, 1, s));
  }
  return ERI_OK;
}

// Density-weighted batch screening (Eq. 8-9 and Alg. 1 lines 12-16): per call, from the density itself,
// P_{ab|cd} = the largest |D| over the six sub-blocks between the four shell groups of a unit; a quartet of the unit is
// evaluated iff Q_ij Q_kl min(1, P_{ab|cd}) >= tau.  All of it runs on the device on the caller's stream (no host
// synchronisation): one pass over D, then one launch that writes each unit's effective threshold, the kept ket prefix
// of every bra pair and the number of surviving quartets.
int dscreen_prepare(eri_plan& pl, const double* D, cudaStream_t s) {
  const Basis& b = pl.basis;
  const int ng = (int)b.groups.size(), nu = (int)pl.units.size();
  if (!pl.ds_ready) {
    std::vector<int> ag(b.nao);
    for (size_t sh = 0; sh < b.sh.size(); ++sh)
      for (int k = 0; k < nsph(b.sh[sh].l); ++k) ag[b.sh[sh].ao_off + k] = b.group_of[sh];
    CK(pl.ao_group.upload(ag, s));
    CK(pl.pmax.alloc((size_t)ng * ng)); CK(pl.ds_kept.alloc(nu)); CK(pl.thr_eff.alloc(nu));
    std::vector<DscreenUnit> du(nu);
    for (int k = 0; k < nu; ++k) {
      Unit& u = *pl.units[k]; const PairClass& P = *pl.pcs[u.P]; const PairClass& R = *pl.pcs[u.R];
      CK(u.ket_count_dyn.alloc(P.npair));
      du[k] = DscreenUnit{P.q.p, R.q.p, u.ket_count.p, u.ket_count_dyn.p, P.npair, {P.ga, P.gb, R.ga, R.gb}};
      pl.ds_max_nbra = std::max(pl.ds_max_nbra, P.npair);
    }
    CK(pl.ds_units.upload(du, s));
    CK(cudaStreamSynchronize(s));   // the host vectors die here (first call only)
    pl.ds_ready = true;
  }
  CK(cudaMemsetAsync(pl.pmax.p, 0, sizeof(unsigned long long) * ng * ng, s));
  CK(cudaMemsetAsync(pl.ds_kept.p, 0, sizeof(unsigned long long) * nu, s));
  CK(launch_group_max(D, b.nao, pl.ao_group.p, ng, pl.pmax.p, s));
  CK(launch_dscreen(pl.ds_units.p, nu, pl.ds_max_nbra, pl.pmax.p, ng, pl.thr, pl.thr_eff.p, pl.ds_kept.p, s));
  return ERI_OK;
}

int jk_grad(eri_plan& pl, const double* D, double* gJ, double* gK, cudaStream_t s) {
  if (!D || !gJ || !gK) return fail(ERI_ERR_BAD_ARG, "null pointer");
  if (pl.is_list || !pl.want_grad) return fail(ERI_ERR_BAD_ARG, "plan was not created with want_grad");
  CKI(ensure_init());   // device check
  if (pl.basis.natm == 0) return ERI_OK;
  CK(cudaMemsetAsync(gJ, 0, sizeof(double) * 3 * pl.basis.natm, s));
  CK(cudaMemsetAsync(gK, 0, sizeof(double) * 3 * pl.basis.natm, s));
  if (pl.basis.nao == 0) return ERI_OK;
  CK(launch_sph2cart(pl.map, D, pl.Dc.p, s));
  return run_units(pl, true, gJ, gK, s);
}

}  // namespace
}  // namespace eri

// =================================================================================================================
extern "C" {

const char* eri_version(void) { return "liberi_b200 0.1 (sm_100a)"; }
const char* eri_last_error(void) { return g_err.c_str(); }
const char* eri_strerror(int code) {
  switch (code) {
    case ERI_OK: return "ok";
    case ERI_ERR_BAD_ARG: return "bad argument";
    case ERI_ERR_UNSUPPORTED_L: return "angular momentum outside 0..6";
    case ERI_ERR_CUDA: return "CUDA failure";
    case ERI_ERR_NOMEM: return "out of memory";
    default: return "unknown error code";
  }
}

double eri_canonical_flops(int la, int lb, int lc, int ld, int ka, int kb, int kc, int kd, int deriv) {
  return canonical_flops(la, lb, lc, ld, ka, kb, kc, kd, deriv);
}

int eri_plan_create(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim, const double* coords, int natm,
                    double schwarz_thr, int want_grad, void* stream, eri_plan_t** out) {
  if (!out) return fail(ERI_ERR_BAD_ARG, "null out pointer");
  *out = nullptr;
  try {
    auto pl = std::make_unique<eri_plan>();
    CKI(create_dense_plan(shells, nshell, prims, nprim, coords, natm, schwarz_thr, want_grad, (cudaStream_t)stream, *pl));
    *out = pl.release();
    return ERI_OK;
  } catch (const std::bad_alloc&) { return fail(ERI_ERR_NOMEM, "host allocation failed"); }
    catch (...) { return fail(ERI_ERR_BAD_ARG, "unexpected exception"); }
}

int eri_list_plan_create(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim, const double* coords, int natm,
                         const int32_t* quartets, int n, void* stream, eri_plan_t** out) {
  if (!out) return fail(ERI_ERR_BAD_ARG, "null out pointer");
  *out = nullptr;
  try {
    auto pl = std::make_unique<eri_plan>();
    CKI(create_list_plan(shells, nshell, prims, nprim, coords, natm, quartets, n, (cudaStream_t)stream, *pl, nullptr, nullptr));
    *out = pl.release();
    return ERI_OK;
  } catch (const std::bad_alloc&) { return fail(ERI_ERR_NOMEM, "host allocation failed"); }
    catch (...) { return fail(ERI_ERR_BAD_ARG, "unexpected exception"); }
}

void eri_plan_destroy(eri_plan_t* plan) {
  if (!plan) return;
  cudaDeviceSynchronize();   // the plan's buffers go back to the allocator's pool: nothing may still be using them
  delete plan;
}
int eri_plan_set_shard(eri_plan_t* plan, int rank, int nranks) {
  if (!plan || nranks < 1 || rank < 0 || rank >= nranks) return fail(ERI_ERR_BAD_ARG, "bad shard %d of %d", rank, nranks);
  plan->shard = rank; plan->nshard = nranks; ++plan->sel_gen;
  return ERI_OK;
}

int eri_plan_build_jk(eri_plan_t* plan, const double* D, double* J, double* K, void* stream) {
  if (!plan) return fail(ERI_ERR_BAD_ARG, "null plan");
  if (plan->is_list) return fail(ERI_ERR_BAD_ARG, "list plan: use eri_list_plan_digest");
  return build_jk(*plan, D, J, K, (cudaStream_t)stream);
}
int eri_list_plan_digest(eri_plan_t* plan, const double* D, double* Jt, double* Kt, void* stream) {
  if (!plan) return fail(ERI_ERR_BAD_ARG, "null plan");
  if (!plan->is_list) return fail(ERI_ERR_BAD_ARG, "not a list plan");
  return build_jk(*plan, D, Jt, Kt, (cudaStream_t)stream);
}
int eri_plan_jk_grad(eri_plan_t* plan, const double* D, double* gJ, double* gK, void* stream) {
  if (!plan) return fail(ERI_ERR_BAD_ARG, "null plan");
  return jk_grad(*plan, D, gJ, gK, (cudaStream_t)stream);
}

int eri_plan_build_jk_dscreen(eri_plan_t* plan, const double* D, double* J, double* K, void* stream) {
  if (!plan || !D || !J || !K) return fail(ERI_ERR_BAD_ARG, "null pointer");
  if (plan->is_list) return fail(ERI_ERR_BAD_ARG, "list plan: density-weighted screening needs a dense plan");
  if (!(plan->thr > 0.0)) return eri_plan_build_jk(plan, D, J, K, stream);   // tau = 0: nothing is ever skipped
  CKI(ensure_init());
  if (plan->basis.nao == 0) return ERI_OK;
  CKI(dscreen_prepare(*plan, D, (cudaStream_t)stream));
  plan->ds_active = true;
  const int rc = build_jk(*plan, D, J, K, (cudaStream_t)stream);
  plan->ds_active = false;
  return rc;
}
int eri_plan_dscreen_quartets(eri_plan_t* plan, int64_t* out) {
  if (!plan || !out) return fail(ERI_ERR_BAD_ARG, "null pointer");
  *out = 0;
  if (!plan->ds_ready) return ERI_OK;
  std::vector<unsigned long long> h(plan->units.size());
  CK(cudaMemcpy(h.data(), plan->ds_kept.p, sizeof(unsigned long long) * h.size(), cudaMemcpyDeviceToHost));
  for (unsigned long long v : h) *out += (int64_t)v;
  return ERI_OK;
}

int eri_plan_dscreen_group_max(eri_plan_t* plan, int32_t* ao_group, double* P) {
  if (!plan) return fail(ERI_ERR_BAD_ARG, "null plan");
  if (!plan->ds_ready) return fail(ERI_ERR_BAD_ARG, "no density-weighted build has run on this plan");
  const size_t ng = plan->basis.groups.size();
  CK(cudaDeviceSynchronize());
  if (ao_group) CK(cudaMemcpy(ao_group, plan->ao_group.p, sizeof(int) * plan->basis.nao, cudaMemcpyDeviceToHost));
  if (P) {
    std::vector<unsigned long long> h(ng * ng);
    CK(cudaMemcpy(h.data(), plan->pmax.p, sizeof(unsigned long long) * h.size(), cudaMemcpyDeviceToHost));
    std::memcpy(P, h.data(), sizeof(double) * h.size());   // the accumulators hold the bit patterns of non-negative doubles
  }
  return ERI_OK;
}

// Allocation-free: must not reach ensure_init (it allocates the Rys buffer on its first call) or any Dev<>::alloc.
int eri_density_group_max_noalloc(const double* D, int nao, const int32_t* ao_group, int ngroups, double* P, void* stream) {
  if (nao < 0 || ngroups < 0) return fail(ERI_ERR_BAD_ARG, "negative size (nao %d, ngroups %d)", nao, ngroups);
  if (ngroups > ERI_NOALLOC_MAX_GROUPS)
    return fail(ERI_ERR_BAD_ARG, "ngroups %d exceeds ERI_NOALLOC_MAX_GROUPS = %d, the size of the static scratch array", ngroups, ERI_NOALLOC_MAX_GROUPS);
  if (ngroups == 0) return ERI_OK;
  if (!P || (nao > 0 && (!D || !ao_group))) return fail(ERI_ERR_BAD_ARG, "null pointer");
  CK(launch_group_max_noalloc(D, nao, ao_group, ngroups, P, (cudaStream_t)stream));
  return ERI_OK;
}

int eri_plan_build_jk_host(eri_plan_t* plan, const double* D, double* J, double* K, void* stream) {
  if (!plan || !D || !J || !K) return fail(ERI_ERR_BAD_ARG, "null pointer");
  cudaStream_t s = (cudaStream_t)stream;
  const size_t n2 = (size_t)plan->basis.nao * plan->basis.nao;
  if (plan->Dh.n != n2) { CK(plan->Dh.alloc(n2)); CK(plan->Jh.alloc(n2)); CK(plan->Kh.alloc(n2)); }
  CK(cudaMemcpyAsync(plan->Dh.p, D, n2 * sizeof(double), cudaMemcpyHostToDevice, s));
  CKI(plan->is_list ? eri_list_plan_digest(plan, plan->Dh.p, plan->Jh.p, plan->Kh.p, stream)
                    : eri_plan_build_jk(plan, plan->Dh.p, plan->Jh.p, plan->Kh.p, stream));
  CK(cudaMemcpyAsync(J, plan->Jh.p, n2 * sizeof(double), cudaMemcpyDeviceToHost, s));
  CK(cudaMemcpyAsync(K, plan->Kh.p, n2 * sizeof(double), cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  return ERI_OK;
}

int eri_plan_jk_grad_host(eri_plan_t* plan, const double* D, double* gJ, double* gK, void* stream) {
  if (!plan || !D || !gJ || !gK) return fail(ERI_ERR_BAD_ARG, "null pointer");
  cudaStream_t s = (cudaStream_t)stream;
  const size_t n2 = (size_t)plan->basis.nao * plan->basis.nao, ng = 3 * (size_t)plan->basis.natm;
  if (plan->Dh.n != n2) { CK(plan->Dh.alloc(n2)); CK(plan->Jh.alloc(n2)); CK(plan->Kh.alloc(n2)); }
  if (plan->gJd.n != ng) { CK(plan->gJd.alloc(ng)); CK(plan->gKd.alloc(ng)); }
  CK(cudaMemcpyAsync(plan->Dh.p, D, n2 * sizeof(double), cudaMemcpyHostToDevice, s));
  CKI(eri_plan_jk_grad(plan, plan->Dh.p, plan->gJd.p, plan->gKd.p, stream));
  CK(cudaMemcpyAsync(gJ, plan->gJd.p, ng * sizeof(double), cudaMemcpyDeviceToHost, s));
  CK(cudaMemcpyAsync(gK, plan->gKd.p, ng * sizeof(double), cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  return ERI_OK;
}

int eri_plan_stats(const eri_plan_t* plan, eri_stats_t* out) {
  if (!plan || !out) return fail(ERI_ERR_BAD_ARG, "null pointer");
  *out = plan->stats;
  return ERI_OK;
}
int eri_plan_num_classes(const eri_plan_t* plan) { return plan ? (int)plan->units.size() : ERI_ERR_BAD_ARG; }
int eri_plan_class_stats(const eri_plan_t* cplan, eri_class_stat_t* out, int max_entries) {
  if (!cplan || (!out && max_entries > 0)) return fail(ERI_ERR_BAD_ARG, "null pointer");
  eri_plan_t* plan = const_cast<eri_plan_t*>(cplan);
  if (plan->ev_pending) {   // collect the per-unit device times of the last timed call
    const size_t n = plan->units.size();
    CK(cudaEventSynchronize(plan->ev[n]));
    for (size_t u = 0; u < n; ++u) {
      float ms = 0; CK(cudaEventElapsedTime(&ms, plan->ev[u], plan->ev[u + 1]));
      (plan->ev_grad ? plan->units[u]->last_ms_grad : plan->units[u]->last_ms) = ms;
    }
    plan->ev_pending = false;
  }
  int k = 0;
  for (const auto& up : plan->units) {
    if (k >= max_entries) break;
    const Unit& u = *up; const PairClass& P = *plan->pcs[u.P]; const PairClass& R = *plan->pcs[u.R];
    eri_class_stat_t& c = out[k++];
    c.la = P.la; c.lb = P.lb; c.lc = R.la; c.ld = R.lb; c.ka = P.Ka; c.kb = P.Kb; c.kc = R.Ka; c.kd = R.Kb;
    c.nroots = (P.la + P.lb + R.la + R.lb) / 2 + 1; c.kernel = u.kernel; c.quartets = u.quartets;
    c.slots = plan->is_list ? u.quartets : u.kernel == 3 ? u.t_slots : (long long)u.nblocks * u.BI * u.BJ;
    c.canonical_flops = u.flops; c.last_ms = u.last_ms; c.last_ms_grad = u.last_ms_grad;
    c.kernel_grad = u.kernel_grad; c.canonical_flops_grad = u.flops_grad;
    c.tile_fill_pm = u.t_slots > 0 ? (int)(1000.0 * (double)u.quartets / (double)u.t_slots + 0.5) : 0;
  }
  return k;
}
int eri_plan_set_timing(eri_plan_t* plan, int on) { if (!plan) return fail(ERI_ERR_BAD_ARG, "null plan"); plan->timing = on; return ERI_OK; }
static int reselect_kernels(eri_plan_t* plan) {
  // host-synchronous like plan creation: waits for the device (the plan's launches in flight), then uploads the row tables
  // of the new selection on a private stream
  CK(cudaDeviceSynchronize());   // the old row tables are released below: no launch may still be reading them
  cudaStream_t st = nullptr;
  CK(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
  int rc = ERI_OK;
  for (auto& u : plan->units) { rc = select_kernels(*plan, *u, st); if (rc != ERI_OK) break; }
  cudaStreamSynchronize(st); cudaStreamDestroy(st);
  plan->order.clear(); plan->order_grad.clear(); ++plan->sel_gen;
  return rc;
}
int eri_plan_set_kernel_mode(eri_plan_t* plan, int mode) {
  if (!plan || mode < 0 || mode > 2) return fail(ERI_ERR_BAD_ARG, "bad kernel mode");
  CKI(ensure_init());   // device check
  plan->kernel_mode = mode;
  return reselect_kernels(plan);
}
int eri_plan_set_tuning(eri_plan_t* plan, int key, double value) {
  if (!plan || !(value >= 0.0)) return fail(ERI_ERR_BAD_ARG, "bad tuning value");
  CKI(ensure_init());
  if (key == ERI_TUNE_TILE_FILL_SCALE) plan->tile_fill_scale = value;
  else if (key == ERI_TUNE_GRAD_MIN_TASKS) plan->grad_min_tasks = (long long)value;
  else if (key == ERI_TUNE_PGRAD_MIN_NPP) plan->pgrad_min_npp = (long long)value;
  else return fail(ERI_ERR_BAD_ARG, "unknown tuning key %d", key);
  return reselect_kernels(plan);
}
int eri_kernel_catalog(char* buf, int n) {
  std::vector<std::string> v; tuned_catalog(v);
  std::string all; for (const std::string& x : v) { all += x; all += '\n'; }
  if (buf && n > 0) { const size_t m = std::min((size_t)n - 1, all.size()); std::memcpy(buf, all.data(), m); buf[m] = 0; }
  return (int)all.size() + 1;
}
int eri_kernel_launched(char* buf, int n) {
  std::string all;
  { std::lock_guard<std::mutex> lk(g_log_mu); for (const std::string& x : g_launched) { all += x; all += '\n'; } }
  if (buf && n > 0) { const size_t m = std::min((size_t)n - 1, all.size()); std::memcpy(buf, all.data(), m); buf[m] = 0; }
  return (int)all.size() + 1;
}

int eri_build_jk(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim, const double* coords, int natm,
                 const double* D, double schwarz_thr, double* J, double* K, void* stream) {
  eri_plan_t* pl = nullptr;
  CKI(eri_plan_create(shells, nshell, prims, nprim, coords, natm, schwarz_thr, 0, stream, &pl));
  int r = eri_plan_build_jk(pl, D, J, K, stream);
  if (r == ERI_OK && cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) r = fail(ERI_ERR_CUDA, "stream synchronise failed");
  eri_plan_destroy(pl);
  return r;
}

int eri_jk_grad(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim, const double* coords, int natm,
                const double* D, double schwarz_thr, double* gJ, double* gK, void* stream) {
  eri_plan_t* pl = nullptr;
  CKI(eri_plan_create(shells, nshell, prims, nprim, coords, natm, schwarz_thr, 1, stream, &pl));
  int r = eri_plan_jk_grad(pl, D, gJ, gK, stream);
  if (r == ERI_OK && cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) r = fail(ERI_ERR_CUDA, "stream synchronise failed");
  eri_plan_destroy(pl);
  return r;
}

int eri_digest_quartet_list(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim, const double* coords, int natm,
                            const int32_t* quartets, int n, const double* D, double* Jt, double* Kt, void* stream) {
  eri_plan_t* pl = nullptr;
  CKI(eri_list_plan_create(shells, nshell, prims, nprim, coords, natm, quartets, n, stream, &pl));
  int r = eri_list_plan_digest(pl, D, Jt, Kt, stream);
  if (r == ERI_OK && cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) r = fail(ERI_ERR_CUDA, "stream synchronise failed");
  eri_plan_destroy(pl);
  return r;
}

int eri_compute_quartets(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim, const double* coords, int natm,
                         const int32_t* quartets, int n, double* out, const int64_t* out_off, void* stream) {
  if (n == 0) return ERI_OK;
  if (!out || !out_off) return fail(ERI_ERR_BAD_ARG, "null output pointer");
  cudaStream_t s = (cudaStream_t)stream;
  try {
    eri_plan pl;
    std::vector<long long> coff; long long ctot = 0;
    CKI(create_list_plan(shells, nshell, prims, nprim, coords, natm, quartets, n, s, pl, &coff, &ctot));
    Dev<double> cart; CK(cart.alloc((size_t)ctot));
    CK(cudaMemsetAsync(cart.p, 0, sizeof(double) * (size_t)ctot, s));
    for (auto& up : pl.units) {
      Work w = make_work(pl, *up, false);
      CK(launch_generic_store(w, cart.p, up->coff.p, 1, s));
    }
    std::vector<int> q4(quartets, quartets + 4 * (size_t)n);
    std::vector<long long> ooff(out_off, out_off + n);
    Dev<int> dq4; Dev<long long> dcoff, dooff;
    CK(dq4.upload(q4, s)); CK(dcoff.upload(coff, s)); CK(dooff.upload(ooff, s));
    CK(launch_block_c2s(pl.map, dq4.p, n, cart.p, dcoff.p, out, dooff.p, s));
    CK(cudaStreamSynchronize(s));
    return ERI_OK;
  } catch (const std::bad_alloc&) { return fail(ERI_ERR_NOMEM, "host allocation failed"); }
}

int eri_schwarz(const eri_shell_t* shells, int nshell, const eri_prim_t* prims, int nprim, const double* coords, int natm,
                double* Q, void* stream) {
  if (!Q && nshell > 0) return fail(ERI_ERR_BAD_ARG, "null output pointer");
  cudaStream_t s = (cudaStream_t)stream;
  try {
    Basis b;
    CKI(make_basis(shells, nshell, prims, nprim, coords, natm, b));
    CKI(ensure_init());
    const int ng = (int)b.groups.size();
    for (int ga = 0; ga < ng; ++ga)
      for (int gb = 0; gb <= ga; ++gb) {
        PairClass pc; init_pair_class(b, ga, gb, pc);
        for (int A : b.groups[ga].shells) for (int B : b.groups[gb].shells) { pc.sa.push_back(A); pc.sb.push_back(B); }
        CKI(upload_pair_class(b, pc, s));
        Dev<double> qd; SchwarzScratch sc;
        CKI(schwarz_enqueue(pc, qd, sc, s));
        CK(cudaStreamSynchronize(s));
        CKI(schwarz_collect(pc, qd));
        for (int i = 0; i < pc.npair; ++i) Q[(size_t)pc.sa[i] * nshell + pc.sb[i]] = Q[(size_t)pc.sb[i] * nshell + pc.sa[i]] = pc.Q[i];
      }
    return ERI_OK;
  } catch (const std::bad_alloc&) { return fail(ERI_ERR_NOMEM, "host allocation failed"); }
}

int eri_rys_roots(int nroots, const double* x, int n, double* u, double* w) {
  if (nroots < 1 || nroots > RYS_NMAX) return fail(ERI_ERR_BAD_ARG, "nroots outside 1..%d", RYS_NMAX);
  if (n < 0 || (n > 0 && (!x || !u || !w))) return fail(ERI_ERR_BAD_ARG, "null pointer");
  if (n == 0) return ERI_OK;
  CKI(ensure_init());
  Dev<double> dx, du, dw;
  std::vector<double> hx(x, x + n);
  CK(dx.upload(hx, nullptr)); CK(du.alloc((size_t)n * nroots)); CK(dw.alloc((size_t)n * nroots));
  CK(launch_rys_diag(nroots, g_rys, dx.p, n, du.p, dw.p, nullptr));
  CK(cudaMemcpy(u, du.p, sizeof(double) * n * nroots, cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(w, dw.p, sizeof(double) * n * nroots, cudaMemcpyDeviceToHost));
  return ERI_OK;
}

int eri_c2s_matrix(int l, double* T) {   // diagnostic: the library's ns(l) x nc(l) table (reading R3)
  if (l < 0 || l > LMAX || !T) return fail(ERI_ERR_BAD_ARG, "bad argument");
  std::vector<double> t; build_c2s(l, t);
  std::memcpy(T, t.data(), sizeof(double) * t.size());
  return ERI_OK;
}

int eri_measure_fp64_peak(double* tflops, void* stream) {
  if (!tflops) return fail(ERI_ERR_BAD_ARG, "null pointer");
  CKI(ensure_init());   // device check
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  CK(cudaGetDevice(&dev)); CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  Dev<double> sink; CK(sink.alloc(1));
  cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  const int blocks = sms * 8, iters = 100000;   // at least 1e5 iterations
  CK(launch_fp64_peak(sink.p, 2000, blocks, s));
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    CK(cudaEventRecord(e0, s)); CK(launch_fp64_peak(sink.p, iters, blocks, s)); CK(cudaEventRecord(e1, s));
    CK(cudaEventSynchronize(e1));
    float ms = 0; CK(cudaEventElapsedTime(&ms, e0, e1));
    best = std::max(best, 2.0 * 16.0 * iters * 256.0 * blocks / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *tflops = best;
  return ERI_OK;
}

}  // extern "C"
