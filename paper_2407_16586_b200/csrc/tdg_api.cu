// tdg_api.cu — C ABI of libtdgrad (include/tdgrad.h): context, host planner (steps a0-a2), density preparation
// and per-class launches (a3-a9).  No CPU arithmetic fallback: all integrals are evaluated by the CUDA kernels.
#include <algorithm>
#include <atomic>
#include <thread>
#include <cmath>
#include <cstring>
#include <map>
#include <new>
#include <string>
#include <vector>

#include "../../include/tdgrad.h"
#include "tdg_grad.cuh"
#include "tdg_internal.h"

#define PCLS(la, lb) ((la) * ((la) + 1) / 2 + (lb))
#define TDG_MAX_STREAMS 8
#define TDG_DEFAULT_STREAMS 6

// Launchers register themselves at load time (one translation unit per class and role, tdg_class.cu).
#define TDG_ROLE_SLOTS 64
static tdg_launch_fn g_launchers[TDG_NCLASS][TDG_ROLE_SLOTS];
static int class_index(int la, int lb, int lc, int ld) {
  const int c1 = PCLS(la, lb), c2 = PCLS(lc, ld);
  return c1 * (c1 + 1) / 2 + c2;
}
void tdg_register_launcher(int la, int lb, int lc, int ld, int role, tdg_launch_fn fn) {
  if (la <= TDG_MAX_L && role >= 0 && role < TDG_ROLE_SLOTS) g_launchers[class_index(la, lb, lc, ld)][role] = fn;
}
tdg_launch_fn tdg_get_launcher(int la, int lb, int lc, int ld, int role) {
  return (role >= 0 && role < TDG_ROLE_SLOTS) ? g_launchers[class_index(la, lb, lc, ld)][role] : nullptr;
}
int tdg_num_roles(int la, int lb, int lc, int ld) {
#define TDG_CLASS(a, b, c, d) \
  if (la == a && lb == b && lc == c && ld == d) return QC<a, b, c, d>::NROLE;
#include "tdg_classes.inc"
#undef TDG_CLASS
  return 0;
}

namespace {

struct Bucket {       // shell pairs of one (la, lb, primitive-pair count), ordered by coarse Schwarz bin, then along a space-filling curve
  int la, lb, npp, n;
  PairHdr* d_hdr = nullptr;
  double* d_prim = nullptr;
  std::vector<double> tilemax;   // largest bound of each 32-pair tile
  std::vector<double> sufmax;    // sufmax[k] = max of the bounds of pairs k.. (non-increasing): kets that may pass a bra form a prefix
};
struct Work {         // one kernel launch: bra bucket x ket bucket
  int b1, b2, cls, nblocks, ntiles;
  int* d_cum = nullptr;
};

}  // namespace

struct tdg_ctx {
  int device = 0;
  std::string err;
  // system
  int natom = 0, nshell = 0, nprim = 0, nbf = 0;
  std::vector<double> xyz, exps, cn;   // cn: contraction coefficient x primitive radial norm x shell norm (a0)
  std::vector<DevShell> shells;
  double *d_xyz = nullptr, *d_exps = nullptr, *d_cn = nullptr, *d_Q = nullptr, *d_rys = nullptr;
  DevShell* d_shells = nullptr;
  int* d_bf2sh = nullptr;
  bool have_Q = false;
  // input basis (tdg_set_spherical): matrices are passed in a basis where flagged d/f shells are real solid harmonics
  bool any_sph = false;
  int nbf_in = 0;
  int *d_inoff = nullptr, *d_sph = nullptr, *d_in2sh = nullptr;
  // plan
  bool planned = false;
  tdg_options opt{};
  std::vector<Bucket> buckets;
  std::vector<Work> work;
  char* d_arena = nullptr;
  int64_t pairs_total = 0, pairs_kept = 0;
  int shard_rank = 0, shard_n = 1;   // tdg_set_shard: this context owns every shard_n-th (launch, bra tile) work item
  int nstreams = 1;                  // tdg_set_streams: the launches of ONE class are dealt over the caller's stream + nstreams-1 side streams
  cudaStream_t side[TDG_MAX_STREAMS - 1] = {};
  cudaEvent_t ev_fork = nullptr, ev_join[TDG_MAX_STREAMS - 1] = {};
  // per-call scratch
  double* d_grad = nullptr;
  double* d_dmax = nullptr;
  unsigned long long* d_counters = nullptr;   // [nwork][3]
  size_t counters_cap = 0;
  std::vector<std::pair<size_t, void*>> scratch;  // cached matrix-sized buffers (bytes, ptr)
  std::vector<bool> scratch_used;
};

// Width of the coarse Schwarz bins of the pair order (tdg_plan): bounds within this factor share a bin.  Measured on cfg 3
// (profiles/r02_pair_order.md): 2, 4 and 16 give the same step time within 0.5 %; 4 costs 14 % more screened candidates than the exact sort.
#define TDG_QBIN_FACTOR 4.0

static int fail_cuda(tdg_ctx* c, cudaError_t e, const char* where) {
  c->err = std::string(where) + ": " + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? TDG_ENOMEM : TDG_ECUDA;
}
#define CK(call)                                                  \
  do {                                                            \
    cudaError_t e_ = (call);                                      \
    if (e_ != cudaSuccess) return fail_cuda(ctx, e_, #call);      \
  } while (0)

static void free_plan(tdg_ctx* c) {
  cudaFree(c->d_arena); c->d_arena = nullptr;   // bucket headers, primitive-pair records and work lists live in one allocation
  c->buckets.clear(); c->work.clear();
  c->planned = false;
}
static void free_system(tdg_ctx* c) {
  free_plan(c);
  cudaFree(c->d_xyz); cudaFree(c->d_exps); cudaFree(c->d_cn); cudaFree(c->d_Q); cudaFree(c->d_shells);
  cudaFree(c->d_grad); cudaFree(c->d_dmax); cudaFree(c->d_bf2sh); c->d_bf2sh = nullptr;
  cudaFree(c->d_inoff); cudaFree(c->d_sph); cudaFree(c->d_in2sh); c->d_inoff = c->d_sph = c->d_in2sh = nullptr;
  c->any_sph = false; c->nbf_in = 0;
  c->d_xyz = c->d_exps = c->d_cn = c->d_Q = c->d_grad = c->d_dmax = nullptr; c->d_shells = nullptr;
  for (auto& s : c->scratch) cudaFree(s.second);
  c->scratch.clear(); c->scratch_used.clear();
  c->have_Q = false; c->nshell = 0; c->natom = 0; c->nbf = 0; c->nprim = 0;
}

extern "C" const char* tdg_strerror(int code) {
  switch (code) {
    case TDG_OK: return "ok";
    case TDG_EINVAL: return "invalid argument";
    case TDG_EUNSUPPORTED: return "unsupported (angular momentum > 3 or class not built)";
    case TDG_ENOTPLANNED: return "tdg_set_system/tdg_plan not called";
    case TDG_ENOMEM: return "out of memory";
    case TDG_ECUDA: return "CUDA error";
  }
  return "unknown error";
}
extern "C" const char* tdg_last_error(const tdg_ctx* ctx) { return ctx ? ctx->err.c_str() : ""; }

extern "C" int tdg_create(tdg_ctx** out, int cuda_device) {
  if (!out) return TDG_EINVAL;
  *out = nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) { cudaGetLastError(); return TDG_ECUDA; }
  if (cudaSetDevice(cuda_device) != cudaSuccess) return TDG_ECUDA;
  tdg_ctx* ctx = new (std::nothrow) tdg_ctx();
  if (!ctx) return TDG_ENOMEM;
  ctx->device = cuda_device;
  if (tdg_upload_rys_table(&ctx->d_rys) != cudaSuccess) { delete ctx; return TDG_ECUDA; }
  *out = ctx;
  if (tdg_set_streams(ctx, TDG_DEFAULT_STREAMS) != TDG_OK) { *out = nullptr; tdg_destroy(ctx); return TDG_ECUDA; }
  return TDG_OK;
}

extern "C" int tdg_destroy(tdg_ctx* ctx) {
  if (!ctx) return TDG_EINVAL;
  cudaSetDevice(ctx->device);
  free_system(ctx);
  cudaFree(ctx->d_rys); cudaFree(ctx->d_counters);
  for (int i = 0; i < TDG_MAX_STREAMS - 1; ++i) {
    if (ctx->side[i]) cudaStreamDestroy(ctx->side[i]);
    if (ctx->ev_join[i]) cudaEventDestroy(ctx->ev_join[i]);
  }
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  delete ctx;
  return TDG_OK;
}

extern "C" int tdg_set_shard(tdg_ctx* ctx, int rank, int nranks) {
  if (!ctx || nranks <= 0 || rank < 0 || rank >= nranks) return TDG_EINVAL;
  if (rank != ctx->shard_rank || nranks != ctx->shard_n) { cudaSetDevice(ctx->device); free_plan(ctx); }
  ctx->shard_rank = rank; ctx->shard_n = nranks;
  return TDG_OK;
}

extern "C" int tdg_set_streams(tdg_ctx* ctx, int nstreams) {
  if (!ctx || nstreams < 1 || nstreams > TDG_MAX_STREAMS) return TDG_EINVAL;
  cudaSetDevice(ctx->device);
  if (!ctx->ev_fork) CK(cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming));
  for (int i = 0; i < nstreams - 1; ++i) {
    if (!ctx->side[i]) CK(cudaStreamCreateWithFlags(&ctx->side[i], cudaStreamNonBlocking));
    if (!ctx->ev_join[i]) CK(cudaEventCreateWithFlags(&ctx->ev_join[i], cudaEventDisableTiming));
  }
  ctx->nstreams = nstreams;
  return TDG_OK;
}

extern "C" int tdg_nbf(const tdg_ctx* ctx, int* nbf) {
  if (!ctx || !nbf) return TDG_EINVAL;
  *nbf = ctx->nbf_in;   // size of the matrices the caller passes (= the Cartesian count unless tdg_set_spherical flagged shells)
  return TDG_OK;
}

// Step a0 (eq 38 "N"; eq 43; O1): coefficient of each primitive =
// d_k (2z/pi)^(3/4) (4z)^(l/2) / sqrt(S), S = sum_kk' d_k d_k' (2 sqrt(z z')/(z+z'))^(l+3/2); the per-component
// factor 1/sqrt((2lx-1)!!(2ly-1)!!(2lz-1)!!) is applied to the density products inside the kernels.
extern "C" int tdg_set_system(tdg_ctx* ctx, int natom, const double* xyz, int nshell, const tdg_shell* shells,
                              int nprim_total, const double* exps, const double* coefs) {
  if (!ctx) return TDG_EINVAL;
  if (!xyz || !shells || !exps || !coefs || natom <= 0 || nshell <= 0 || nprim_total <= 0) return TDG_EINVAL;
  for (int s = 0; s < nshell; ++s) {
    const tdg_shell& sh = shells[s];
    if (sh.atom < 0 || sh.atom >= natom || sh.nprim <= 0 || sh.prim_off < 0 || sh.prim_off + sh.nprim > nprim_total || sh.l < 0) return TDG_EINVAL;
    if (sh.l > TDG_MAX_L) return TDG_EUNSUPPORTED;
    for (int k = 0; k < sh.nprim; ++k) if (!(exps[sh.prim_off + k] > 0.0)) return TDG_EINVAL;
  }
  // a0: all host arithmetic and validation first; the context is only touched once nothing can fail on the host side
  std::vector<double> cn(nprim_total, 0.0);
  std::vector<DevShell> dsh(nshell);
  int off = 0;
  const double PI = 3.14159265358979323846;
  for (int s = 0; s < nshell; ++s) {
    const tdg_shell& sh = shells[s];
    double S = 0.0;
    for (int k = 0; k < sh.nprim; ++k)
      for (int k2 = 0; k2 < sh.nprim; ++k2) {
        const double z1 = exps[sh.prim_off + k], z2 = exps[sh.prim_off + k2];
        S += coefs[sh.prim_off + k] * coefs[sh.prim_off + k2] * std::pow(2.0 * std::sqrt(z1 * z2) / (z1 + z2), sh.l + 1.5);
      }
    if (!(S > 0.0)) return TDG_EINVAL;
    for (int k = 0; k < sh.nprim; ++k) {
      const double z = exps[sh.prim_off + k];
      cn[sh.prim_off + k] = coefs[sh.prim_off + k] * std::pow(2.0 * z / PI, 0.75) * std::pow(4.0 * z, 0.5 * sh.l) / std::sqrt(S);
    }
    dsh[s] = DevShell{sh.atom, sh.l, sh.nprim, sh.prim_off, off, 0};
    off += ncart(sh.l);
  }
  cudaSetDevice(ctx->device);
  free_system(ctx);   // leaves the context empty (nshell = 0): a failed upload below cannot leave a half-initialised system behind
  ctx->xyz.assign(xyz, xyz + 3 * (size_t)natom);
  ctx->exps.assign(exps, exps + nprim_total);
  ctx->cn = std::move(cn);
  ctx->shells = std::move(dsh);
  {
    std::vector<int> bf2sh(off);
    for (int sidx = 0; sidx < nshell; ++sidx)
      for (int f = 0; f < ncart(ctx->shells[sidx].l); ++f) bf2sh[ctx->shells[sidx].bf_off + f] = sidx;
    CK(cudaMalloc(&ctx->d_bf2sh, sizeof(int) * off));
    CK(cudaMemcpy(ctx->d_bf2sh, bf2sh.data(), sizeof(int) * off, cudaMemcpyHostToDevice));
  }
  CK(cudaMalloc(&ctx->d_xyz, sizeof(double) * 3 * natom));
  CK(cudaMalloc(&ctx->d_exps, sizeof(double) * nprim_total));
  CK(cudaMalloc(&ctx->d_cn, sizeof(double) * nprim_total));
  CK(cudaMalloc(&ctx->d_shells, sizeof(DevShell) * nshell));
  CK(cudaMalloc(&ctx->d_Q, sizeof(double) * (size_t)nshell * nshell));
  CK(cudaMalloc(&ctx->d_grad, sizeof(double) * 3 * natom));
  CK(cudaMemcpy(ctx->d_xyz, ctx->xyz.data(), sizeof(double) * 3 * natom, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(ctx->d_exps, ctx->exps.data(), sizeof(double) * nprim_total, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(ctx->d_cn, ctx->cn.data(), sizeof(double) * nprim_total, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(ctx->d_shells, ctx->shells.data(), sizeof(DevShell) * nshell, cudaMemcpyHostToDevice));
  // only now does the context count as holding a system (tdg_plan / tdg_schwarz check nshell > 0)
  ctx->natom = natom; ctx->nshell = nshell; ctx->nprim = nprim_total; ctx->nbf = off; ctx->nbf_in = off;
  return TDG_OK;
}

// NEXT-2: flagged d and f shells enter and leave the library as real solid harmonics.
extern "C" int tdg_set_spherical(tdg_ctx* ctx, const int32_t* spherical) {
  if (!ctx) return TDG_EINVAL;
  if (ctx->nshell <= 0) return TDG_ENOTPLANNED;
  cudaSetDevice(ctx->device);
  const int ns = ctx->nshell;
  std::vector<int> flag(ns, 0), inoff(ns, 0), in2sh;
  bool any = false;
  int off = 0;
  for (int s = 0; s < ns; ++s) {
    const int l = ctx->shells[s].l;
    flag[s] = (spherical && spherical[s] && l >= 2) ? 1 : 0;
    any = any || flag[s];
    inoff[s] = off;
    const int nf = flag[s] ? 2 * l + 1 : ncart(l);
    for (int f = 0; f < nf; ++f) in2sh.push_back(s);
    off += nf;
  }
  cudaFree(ctx->d_inoff); cudaFree(ctx->d_sph); cudaFree(ctx->d_in2sh); ctx->d_inoff = ctx->d_sph = ctx->d_in2sh = nullptr;
  ctx->any_sph = false; ctx->nbf_in = ctx->nbf;
  if (!any) return TDG_OK;
  CK(cudaMalloc(&ctx->d_inoff, sizeof(int) * ns)); CK(cudaMalloc(&ctx->d_sph, sizeof(int) * ns)); CK(cudaMalloc(&ctx->d_in2sh, sizeof(int) * off));
  CK(cudaMemcpy(ctx->d_inoff, inoff.data(), sizeof(int) * ns, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(ctx->d_sph, flag.data(), sizeof(int) * ns, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(ctx->d_in2sh, in2sh.data(), sizeof(int) * off, cudaMemcpyHostToDevice));
  ctx->any_sph = true; ctx->nbf_in = off;
  return TDG_OK;
}

static int ensure_schwarz(tdg_ctx* ctx) {
  if (ctx->have_Q) return TDG_OK;
  CK(tdg_launch_schwarz(ctx->d_shells, ctx->nshell, ctx->d_xyz, ctx->d_exps, ctx->d_cn, ctx->d_rys, ctx->d_Q, 0));
  CK(cudaDeviceSynchronize());
  ctx->have_Q = true;
  return TDG_OK;
}

extern "C" int tdg_schwarz(tdg_ctx* ctx, double* Q_host) {
  if (!ctx || !Q_host) return TDG_EINVAL;
  if (ctx->nshell <= 0) return TDG_ENOTPLANNED;
  cudaSetDevice(ctx->device);
  int rc = ensure_schwarz(ctx);
  if (rc) return rc;
  CK(cudaMemcpy(Q_host, ctx->d_Q, sizeof(double) * (size_t)ctx->nshell * ctx->nshell, cudaMemcpyDeviceToHost));
  return TDG_OK;
}

// Steps a1-a2.
extern "C" int tdg_plan(tdg_ctx* ctx, const tdg_options* opt) {
  if (!ctx) return TDG_EINVAL;
  if (ctx->nshell <= 0) return TDG_ENOTPLANNED;
  cudaSetDevice(ctx->device);
  free_plan(ctx);
  ctx->opt = opt ? *opt : tdg_options{0.0, 0, 0, 0};
  const double tau = ctx->opt.tau;
  const int ns = ctx->nshell;
  std::vector<double> Q;
  double Qmax = 0.0;
  if (tau > 0.0) {
    int rc = ensure_schwarz(ctx);
    if (rc) return rc;
    try { Q.resize((size_t)ns * ns); } catch (...) { return TDG_ENOMEM; }
    CK(cudaMemcpy(Q.data(), ctx->d_Q, sizeof(double) * Q.size(), cudaMemcpyDeviceToHost));
    for (double q : Q) if (q > Qmax) Qmax = q;
  }
  struct HP { int i, j; double Q; uint32_t bin, code; };
  // buckets keyed by (pair class, primitive-pair count); a shell's "type" (l, nprim) decides the key, so the pair loop below
  // only indexes a small table (the loop runs over all nshell^2/2 pairs: 4.7e6 at cfg 3, 7.5e7 at cfg 4)
  std::vector<std::pair<int, int>> types;          // distinct (l, nprim)
  std::vector<int> type_of(ns);
  for (int i = 0; i < ns; ++i) {
    const std::pair<int, int> t(ctx->shells[i].l, ctx->shells[i].nprim);
    size_t k = 0;
    while (k < types.size() && types[k] != t) ++k;
    if (k == types.size()) types.push_back(t);
    type_of[i] = (int)k;
  }
  const int nt = (int)types.size();
  std::map<std::pair<int, int>, int> key2group;    // (pair class, npp) -> group, ordered: bucket order = key order
  std::vector<int> tab((size_t)nt * nt, -1);
  for (int a = 0; a < nt; ++a)
    for (int b = 0; b < nt; ++b) {
      const int la = std::max(types[a].first, types[b].first), lb = std::min(types[a].first, types[b].first);
      key2group[{PCLS(la, lb), types[a].second * types[b].second}] = 0;
    }
  {
    int g = 0;
    for (auto& kv : key2group) kv.second = g++;
    for (int a = 0; a < nt; ++a)
      for (int b = 0; b < nt; ++b) {
        const int la = std::max(types[a].first, types[b].first), lb = std::min(types[a].first, types[b].first);
        tab[(size_t)a * nt + b] = key2group[{PCLS(la, lb), types[a].second * types[b].second}];
      }
  }
  ctx->pairs_total = (int64_t)ns * (ns + 1) / 2;
  ctx->pairs_kept = 0;
  try {
    std::vector<std::vector<HP>> groups(key2group.size());
    for (int i = 0; i < ns; ++i) {
      const int ti = type_of[i], li = ctx->shells[i].l;
      const double* Qi = tau > 0.0 ? &Q[(size_t)i * ns] : nullptr;
      for (int j = 0; j <= i; ++j) {
        double q = 1.0;
        if (Qi) { q = Qi[j]; if (!(q * Qmax >= tau)) continue; }
        // orient: higher l first; ties keep i (the larger index) first
        if (li < ctx->shells[j].l) groups[tab[(size_t)ti * nt + type_of[j]]].push_back(HP{j, i, q, 0u, 0u});
        else groups[tab[(size_t)ti * nt + type_of[j]]].push_back(HP{i, j, q, 0u, 0u});
        ++ctx->pairs_kept;
      }
    }
    // Order every bucket by COARSE Schwarz bin (factor TDG_QBIN_FACTOR in Q, descending; PAPER.md:309 sorts by the bound itself) and,
    // inside a bin, along a Morton curve through the pair midpoints: the 32 bras of a tile and the 128 kets of a chunk are then
    // neighbours in space, so the quartets of a block share density blocks (ik), (il), (jk), (jl) and block maxima (L1 hits,
    // merged gather wavefronts) and have similar Rys arguments, while the kets that can pass the Schwarz test with a tile still
    // form a prefix (bounded through the suffix maxima below; every quartet is tested exactly in the kernels).  Headers,
    // primitive-pair records and work lists go into ONE host arena, uploaded with one allocation and one copy.
    double blo[3] = {1e300, 1e300, 1e300}, bhi[3] = {-1e300, -1e300, -1e300};
    for (int a = 0; a < ctx->natom; ++a)
      for (int d = 0; d < 3; ++d) { blo[d] = std::min(blo[d], ctx->xyz[3 * a + d]); bhi[d] = std::max(bhi[d], ctx->xyz[3 * a + d]); }
    auto spread10 = [](uint32_t x) {   // 10 bits -> every third bit
      x &= 0x3ffu; x = (x | (x << 16)) & 0x030000ffu; x = (x | (x << 8)) & 0x0300f00fu; x = (x | (x << 4)) & 0x030c30c3u; x = (x | (x << 2)) & 0x09249249u;
      return x;
    };
    const double qbin_inv_log = 1.0 / std::log(TDG_QBIN_FACTOR);
    auto align16 = [](size_t x) { return (x + 255) & ~(size_t)255; };   // 256-bit loads of the records need 32 bytes; 256 keeps every array on its own line
    size_t bytes = 0;
    std::vector<size_t> off_hdr, off_prim;
    for (auto& kv : key2group) {
      auto& v = groups[kv.second];
      if (v.empty()) continue;
      double qtop = 0.0;
      for (const HP& h : v) qtop = std::max(qtop, h.Q);
      for (HP& h : v) {
        h.bin = (tau > 0.0 && h.Q > 0.0) ? (uint32_t)std::min(4000.0, std::floor(std::log(qtop / h.Q) * qbin_inv_log)) : 0u;
        uint32_t g[3];
        for (int d = 0; d < 3; ++d) {
          const double mid = 0.5 * (ctx->xyz[3 * ctx->shells[h.i].atom + d] + ctx->xyz[3 * ctx->shells[h.j].atom + d]);
          g[d] = (uint32_t)std::min(1023.0, std::max(0.0, (mid - blo[d]) / (bhi[d] - blo[d] + 1e-9) * 1024.0));
        }
        h.code = spread10(g[0]) | (spread10(g[1]) << 1) | (spread10(g[2]) << 2);
      }
      std::sort(v.begin(), v.end(), [](const HP& x, const HP& y) {
        if (x.bin != y.bin) return x.bin < y.bin;
        if (x.code != y.code) return x.code < y.code;
        if (x.i != y.i) return x.i < y.i;
        return x.j < y.j;
      });
      Bucket B;
      B.la = ctx->shells[v[0].i].l; B.lb = ctx->shells[v[0].j].l; B.npp = kv.first.second; B.n = (int)v.size();
      B.tilemax.assign((v.size() + TDG_WARP - 1) / TDG_WARP, 0.0);
      B.sufmax.resize(v.size());
      for (size_t t = 0; t < v.size(); ++t) B.tilemax[t / TDG_WARP] = std::max(B.tilemax[t / TDG_WARP], v[t].Q);
      for (size_t t = v.size(); t-- > 0;) B.sufmax[t] = std::max(v[t].Q, t + 1 < v.size() ? B.sufmax[t + 1] : 0.0);
      off_hdr.push_back(bytes); bytes = align16(bytes + sizeof(PairHdr) * v.size());
      off_prim.push_back(bytes); bytes = align16(bytes + sizeof(double) * v.size() * (size_t)B.npp * TDG_PRIM_STRIDE);
      ctx->buckets.push_back(std::move(B));
    }
    // work lists: bucket b1 >= b2 (bucket order = (pair class, npp) ascending, so bra class >= ket class)
    const int nb = (int)ctx->buckets.size();
    std::vector<std::vector<int>> cums;
    std::vector<size_t> off_cum;
    int64_t item = 0;   // running index of non-empty (launch, bra tile) work items, dealt round-robin over the ranks
    for (int b1 = 0; b1 < nb; ++b1)
      for (int b2 = 0; b2 <= b1; ++b2) {
        const Bucket& X = ctx->buckets[b1]; const Bucket& Y = ctx->buckets[b2];
        const int ntiles = (X.n + TDG_WARP - 1) / TDG_WARP;
        std::vector<int> cum(ntiles + 1, 0);
        for (int t = 0; t < ntiles; ++t) {
          int klen = Y.n;
          if (tau > 0.0) {   // no ket beyond the prefix can pass the Schwarz test with any bra of the tile
            const double qb = X.tilemax[t];
            klen = (int)(std::partition_point(Y.sufmax.begin(), Y.sufmax.end(), [&](double qk) { return qb * qk >= tau; }) - Y.sufmax.begin());
          }
          if (b1 == b2) klen = std::min(klen, std::min(X.n, (t + 1) * TDG_WARP));
          if (klen > 0 && (item++ % ctx->shard_n) != ctx->shard_rank) klen = 0;   // another rank's tile: no blocks here
          cum[t + 1] = cum[t] + (klen + TDG_KB - 1) / TDG_KB;
        }
        if (cum[ntiles] == 0) continue;
        Work W;
        W.b1 = b1; W.b2 = b2; W.ntiles = ntiles; W.nblocks = cum[ntiles];
        const int c1 = PCLS(X.la, X.lb), c2 = PCLS(Y.la, Y.lb);
        W.cls = c1 * (c1 + 1) / 2 + c2;
        off_cum.push_back(bytes); bytes = align16(bytes + sizeof(int) * cum.size());
        cums.push_back(std::move(cum));
        ctx->work.push_back(W);
      }
    // fill the arena (bucket by bucket on a few host threads: exp() per primitive pair) and upload it
    std::vector<char> host(bytes);
    {
      std::vector<std::thread> pool;
      std::atomic<int> next(0);
      const int nthr = std::max(1u, std::min(8u, std::thread::hardware_concurrency()));
      std::vector<const std::vector<HP>*> bucket_pairs;
      for (auto& kv : key2group) if (!groups[kv.second].empty()) bucket_pairs.push_back(&groups[kv.second]);
      // work units: (bucket, slice of 4096 pairs)
      struct Unit { int b; size_t t0, t1; };
      std::vector<Unit> units;
      for (int b = 0; b < nb; ++b)
        for (size_t t0 = 0; t0 < bucket_pairs[b]->size(); t0 += 4096) units.push_back(Unit{b, t0, std::min(bucket_pairs[b]->size(), t0 + 4096)});
      auto fill = [&]() {
        for (;;) {
          const int u = next.fetch_add(1);
          if (u >= (int)units.size()) return;
          const Bucket& B = ctx->buckets[units[u].b];
          const std::vector<HP>& v = *bucket_pairs[units[u].b];
          PairHdr* hdr = reinterpret_cast<PairHdr*>(host.data() + off_hdr[units[u].b]);
          double* prim = reinterpret_cast<double*>(host.data() + off_prim[units[u].b]);
          for (size_t t = units[u].t0; t < units[u].t1; ++t) {
            const DevShell& sa = ctx->shells[v[t].i]; const DevShell& sb = ctx->shells[v[t].j];
            const double* A = &ctx->xyz[3 * sa.atom]; const double* Bc = &ctx->xyz[3 * sb.atom];
            PairHdr& h = hdr[t];
            double R2 = 0.0;
            for (int d = 0; d < 3; ++d) { h.A[d] = A[d]; h.AB[d] = A[d] - Bc[d]; R2 += h.AB[d] * h.AB[d]; }
            h.Q = v[t].Q; h.ish = v[t].i; h.jsh = v[t].j; h.atomA = sa.atom; h.atomB = sb.atom; h.offA = sa.bf_off; h.offB = sb.bf_off;
            double* pp = prim + t * (size_t)B.npp * TDG_PRIM_STRIDE;
            for (int ka = 0; ka < sa.nprim; ++ka)
              for (int kb = 0; kb < sb.nprim; ++kb) {
                const double a = ctx->exps[sa.prim_off + ka], b = ctx->exps[sb.prim_off + kb], p = a + b;
                double* r = pp + (size_t)(ka * sb.nprim + kb) * TDG_PRIM_STRIDE;
                r[0] = p;
                for (int d = 0; d < 3; ++d) r[1 + d] = (a * A[d] + b * Bc[d]) / p;
                r[4] = ctx->cn[sa.prim_off + ka] * ctx->cn[sb.prim_off + kb] * std::exp(-a * b / p * R2) / p;
                r[5] = a; r[6] = b; r[7] = 1.0 / p;
              }
          }
        }
      };
      for (int t = 1; t < nthr; ++t) pool.emplace_back(fill);
      fill();
      for (auto& th : pool) th.join();
    }
    for (size_t w = 0; w < cums.size(); ++w) std::memcpy(host.data() + off_cum[w], cums[w].data(), sizeof(int) * cums[w].size());
    if (bytes) {
      CK(cudaMalloc(&ctx->d_arena, bytes));
      CK(cudaMemcpy(ctx->d_arena, host.data(), bytes, cudaMemcpyHostToDevice));
    }
    for (int b = 0; b < nb; ++b) {
      ctx->buckets[b].d_hdr = reinterpret_cast<PairHdr*>(ctx->d_arena + off_hdr[b]);
      ctx->buckets[b].d_prim = reinterpret_cast<double*>(ctx->d_arena + off_prim[b]);
    }
    for (size_t w = 0; w < cums.size(); ++w) ctx->work[w].d_cum = reinterpret_cast<int*>(ctx->d_arena + off_cum[w]);
  } catch (const std::bad_alloc&) { free_plan(ctx); return TDG_ENOMEM; }
  const size_t need = ctx->work.size() * 3 + 3;
  if (need > ctx->counters_cap) {
    cudaFree(ctx->d_counters); ctx->d_counters = nullptr;
    CK(cudaMalloc(&ctx->d_counters, sizeof(unsigned long long) * need));
    ctx->counters_cap = need;
  }
  ctx->planned = true;
  return TDG_OK;
}

// ---- per-call density preparation (a3) ----
static void* scratch_get(tdg_ctx* ctx, size_t bytes) {
  for (size_t i = 0; i < ctx->scratch.size(); ++i)
    if (!ctx->scratch_used[i] && ctx->scratch[i].first == bytes) { ctx->scratch_used[i] = true; return ctx->scratch[i].second; }
  void* p = nullptr;
  if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  ctx->scratch.push_back({bytes, p}); ctx->scratch_used.push_back(true);
  return p;
}

namespace {
struct Group { std::vector<int> pairs; std::vector<int> canon; };   // canonical matrix id = 2*unique + (0: sym part, 1: antisym part)
struct EventPool {   // timing events of one call; destroyed on every exit path
  std::vector<cudaEvent_t> v;
  cudaEvent_t get() { cudaEvent_t e = nullptr; if (cudaEventCreate(&e) == cudaSuccess) v.push_back(e); return e; }
  ~EventPool() { for (cudaEvent_t e : v) cudaEventDestroy(e); }
};
struct DevTemp {     // cudaMalloc'ed temporary freed on every exit path
  void* p = nullptr;
  ~DevTemp() { cudaFree(p); }
};
}

// Input matrix (host or device, input basis) -> device pointer to its CARTESIAN nbf x nbf form: upload if needed, then
// D_cart = C^T D C when spherical shells are flagged (NEXT-2).
static int to_device_cart(tdg_ctx* ctx, const double* M, int on_dev, cudaStream_t st, const double** out) {
  const size_t nin = (size_t)ctx->nbf_in, n = (size_t)ctx->nbf;
  const double* src = M;
  if (!on_dev) {
    double* buf = (double*)scratch_get(ctx, sizeof(double) * nin * nin);
    if (!buf) { ctx->err = "device allocation of an input matrix failed"; return TDG_ENOMEM; }
    CK(cudaMemcpyAsync(buf, M, sizeof(double) * nin * nin, cudaMemcpyHostToDevice, st));
    src = buf;
  }
  if (ctx->any_sph) {
    double* cart = (double*)scratch_get(ctx, sizeof(double) * n * n);
    if (!cart) { ctx->err = "device allocation of a back-transformed matrix failed"; return TDG_ENOMEM; }
    CK(tdg_launch_sph_transform(src, cart, (int)n, (int)nin, 0, ctx->d_bf2sh, ctx->d_shells, ctx->d_inoff, ctx->d_sph, st));
    src = cart;
  }
  *out = src;
  return TDG_OK;
}

// The launches of one class (one kernel per role, one launch per bucket pair) are independent: they only add into the output
// and into their own counters.  They are dealt over the caller's stream and nstreams-1 side streams that fork from it before
// the class and join it after, so under-filled launches and tails overlap, roles run side by side, and the CUDA events around
// the class (on the caller's stream) time exactly that class.  role_base: 0 gradient kernels, TDG_FOCK_ROLE_BASE Fock kernels.
static int launch_classes(tdg_ctx* ctx, KParams& P, int role_base, double* d_E, bool count_here, cudaStream_t st, EventPool* pool,
                          std::vector<cudaEvent_t>& evs, std::vector<int>& ev_cls, int& launches) {
  const size_t nw = ctx->work.size();
  const int nstr = d_E ? 1 : ctx->nstreams;
  // With per-class timing (stats requested) the side streams join the caller's stream after every class, so that the events time
  // exactly that class; without it they fork once before the first class and join once after the last, and the tail of one class
  // overlaps the start of the next (the tails are the part of a call that does not shrink when the work is sharded over ranks).
  // Measured on cfg 3 (profiles/r02_shard_balance_cfg3.md): free-running is 13 % faster on a 1/8 shard, 5 % on a 1/4 shard, and
  // 1.7 % SLOWER on the whole problem (kernels of different classes then share the SMs for longer), so it is used for shards only.
  const bool join_per_class = pool != nullptr || nstr == 1 || ctx->shard_n == 1;
  std::vector<size_t> order(nw);
  for (size_t w = 0; w < nw; ++w) order[w] = w;
  std::stable_sort(order.begin(), order.end(), [&](size_t x, size_t y) { return ctx->work[x].cls < ctx->work[y].cls; });
  for (size_t g0 = 0; g0 < nw;) {
    size_t g1 = g0;
    while (g1 < nw && ctx->work[order[g1]].cls == ctx->work[order[g0]].cls) ++g1;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (pool) { e0 = pool->get(); e1 = pool->get(); if (!e0 || !e1) return TDG_ECUDA; cudaEventRecord(e0, st); }
    if (nstr > 1 && (join_per_class || g0 == 0)) {
      CK(cudaEventRecord(ctx->ev_fork, st));
      for (int i = 0; i < nstr - 1; ++i) CK(cudaStreamWaitEvent(ctx->side[i], ctx->ev_fork, 0));
    }
    int unit = join_per_class ? 0 : (int)g0;   // free-running: keep dealing round-robin across the class boundary
    for (size_t gw = g0; gw < g1; ++gw) {
      const size_t w = order[gw];
      const Work& W = ctx->work[w];
      const Bucket& X = ctx->buckets[W.b1]; const Bucket& Y = ctx->buckets[W.b2];
      P.bra_hdr = X.d_hdr; P.bra_prim = X.d_prim; P.nbra = X.n; P.nppb = X.npp;
      P.ket_hdr = Y.d_hdr; P.ket_prim = Y.d_prim; P.nket = Y.n; P.nppk = Y.npp;
      P.cum = W.d_cum; P.ntiles = W.ntiles; P.same_bucket = (W.b1 == W.b2) ? 1 : 0;
      P.counters = ctx->d_counters + 3 * (count_here ? w : nw);   // quartet counts come from the first pass only
      if (d_E) { CK(tdg_launch_energy(P, X.la, X.lb, Y.la, Y.lb, W.nblocks, d_E, st)); ++launches; continue; }
      const int nrole = tdg_num_roles(X.la, X.lb, Y.la, Y.lb);
      for (int role = 0; role < nrole; ++role) {   // the roles of a class are separate kernels (slices of the bra function pairs)
        tdg_launch_fn fn = tdg_get_launcher(X.la, X.lb, Y.la, Y.lb, role + role_base);
        if (!fn) { ctx->err = "class kernel not built"; return TDG_EUNSUPPORTED; }
        const int si = unit++ % nstr;
        fn(P, W.nblocks, si == 0 ? st : ctx->side[si - 1]);
        ++launches;
      }
    }
    if (nstr > 1 && (join_per_class || g1 == nw))
      for (int i = 0; i < nstr - 1; ++i) { CK(cudaEventRecord(ctx->ev_join[i], ctx->side[i])); CK(cudaStreamWaitEvent(st, ctx->ev_join[i], 0)); }
    if (pool) { cudaEventRecord(e1, st); evs.push_back(e0); evs.push_back(e1); ev_cls.push_back(ctx->work[order[g0]].cls); }
    g0 = g1;
  }
  return TDG_OK;
}

static int run_contraction(tdg_ctx* ctx, int npair, const double* const* A, const double* const* B, int on_dev,
                           const double* wJ, const double* wK, double cJ, double cK, double cLR, double omega,
                           cudaStream_t st, tdg_stats* stats, double* E_host = nullptr) {
  const int n = ctx->nbf;
  const size_t mbytes = sizeof(double) * (size_t)n * n;
  std::fill(ctx->scratch_used.begin(), ctx->scratch_used.end(), false);
  EventPool pool;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr, ev2 = nullptr;
  if (stats) { ev0 = pool.get(); ev1 = pool.get(); ev2 = pool.get(); if (!ev0 || !ev1 || !ev2) return TDG_ECUDA; cudaEventRecord(ev0, st); }
  // unique input matrices -> device pointers
  std::vector<const double*> uniq, udev;
  auto uid = [&](const double* M) { for (size_t i = 0; i < uniq.size(); ++i) if (uniq[i] == M) return (int)i; return -1; };
  for (int k = 0; k < npair; ++k)
    for (const double* M : {A[k], B[k]}) {
      if (uid(M) >= 0) continue;
      const double* d = nullptr;
      const int rc_in = to_device_cart(ctx, M, on_dev, st, &d);
      if (rc_in) return rc_in;
      uniq.push_back(M); udev.push_back(d);
    }
  if (uniq.size() > 16) return TDG_EINVAL;
  // which inputs are nonsymmetric (their antisymmetric part takes a slot; reading R1 of DESIGN.md)
  double as[16];
  {
    double* d_as = (double*)scratch_get(ctx, 256);
    if (!d_as) return TDG_ENOMEM;
    CK(cudaMemsetAsync(d_as, 0, 256, st));
    for (size_t i = 0; i < uniq.size(); ++i) CK(tdg_launch_asym(udev[i], n, d_as + i, st));
    CK(cudaMemcpyAsync(as, d_as, sizeof(double) * uniq.size(), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
  }
  const bool useK = (cK != 0.0 || cLR != 0.0);
  // groups of density pairs whose canonical matrices fit the 4 slots of the packed array
  std::vector<Group> groups;
  double CJ = 0.0, CKs = 0.0;
  for (int k = 0; k < npair; ++k) {
    CJ += std::fabs(wJ[k] * cJ); CKs += std::fabs(wK[k]);
    const bool doJ = wJ[k] * cJ != 0.0, doK = wK[k] != 0.0 && useK;
    if (!doJ && !doK) continue;
    const int ua = uid(A[k]), ub = uid(B[k]);
    std::vector<int> need = {2 * ua, 2 * ub};
    if (doK && as[ua] != 0.0 && as[ub] != 0.0) { need.push_back(2 * ua + 1); need.push_back(2 * ub + 1); }
    auto merged = [&](const std::vector<int>& base) {
      std::vector<int> r = base;
      for (int c : need) if (std::find(r.begin(), r.end(), c) == r.end()) r.push_back(c);
      return r;
    };
    if (groups.empty() || merged(groups.back().canon).size() > 4) groups.push_back(Group{});
    groups.back().canon = merged(groups.back().canon);
    groups.back().pairs.push_back(k);
  }
  CKs *= std::fabs(cK) + std::fabs(cLR);
  KParams P{};
  P.CJ = CJ; P.CK = CKs;
  P.tau = ctx->opt.tau; P.density_weighted = (ctx->opt.tau > 0.0) ? ctx->opt.density_weighted : 0;
  P.nshell = ctx->nshell; P.sample_mod = ctx->opt.sample_mod; P.sample_seed = ctx->opt.sample_seed;
  P.nbf = n; P.cK = cK; P.cLR = cLR; P.omega = omega; P.omega2 = omega * omega; P.use_lr = (cLR != 0.0) ? 1 : 0;
  P.grad = ctx->d_grad; P.rys_tab = ctx->d_rys;
  int aux_launches = (int)uniq.size();
  if (P.density_weighted) {   // d_ij over ALL input matrices (reading S9)
    if (!ctx->d_dmax) CK(cudaMalloc(&ctx->d_dmax, sizeof(double) * (size_t)ctx->nshell * ctx->nshell));
    MatList ml{};
    ml.n = (int)udev.size();
    for (int i = 0; i < ml.n; ++i) ml.m[i] = udev[i];
    CK(tdg_launch_dmax(ml, n, ctx->d_shells, ctx->nshell, ctx->d_dmax, st));
    P.dmax = ctx->d_dmax;
    aux_launches += 2;
  }
  double* d_E = nullptr;
  if (E_host) {   // energy mode (tdg_energy): same screening and work lists, undifferentiated integrals
    d_E = (double*)scratch_get(ctx, 264);
    if (!d_E) return TDG_ENOMEM;
    CK(cudaMemsetAsync(d_E, 0, sizeof(double), st));
  }
  double* pk = (double*)scratch_get(ctx, 4 * mbytes);
  if (!pk) { ctx->err = "device allocation of the packed density array failed"; return TDG_ENOMEM; }
  P.pk = pk;
  const size_t nw = ctx->work.size();
  CK(cudaMemsetAsync(ctx->d_grad, 0, sizeof(double) * 3 * ctx->natom, st));
  CK(cudaMemsetAsync(ctx->d_counters, 0, sizeof(unsigned long long) * (nw * 3 + 3), st));
  if (stats) cudaEventRecord(ev1, st);
  int launches = 0;
  std::vector<cudaEvent_t> evs;   // (start, stop) per launch, on the launch's own stream
  std::vector<int> ev_cls;
  for (size_t gi = 0; gi < groups.size(); ++gi) {
    const Group& G = groups[gi];
    PackSrc ps{};
    for (size_t m = 0; m < G.canon.size(); ++m) { ps.src[m] = udev[G.canon[m] / 2]; ps.kind[m] = G.canon[m] & 1; }
    CK(tdg_launch_pack(ps, n, ctx->d_bf2sh, ctx->d_shells, pk, st));
    ++aux_launches;
    auto slot = [&](int c) { return (int)(std::find(G.canon.begin(), G.canon.end(), c) - G.canon.begin()); };
    for (int t = 0; t < 16; ++t) { P.MJ[t] = 0.0; P.MK[t] = 0.0; }
    for (int k : G.pairs) {
      const int ua = uid(A[k]), ub = uid(B[k]);
      const int sa = slot(2 * ua), sb = slot(2 * ub);
      const double wj = 4.0 * wJ[k] * cJ, wk = useK ? -2.0 * wK[k] : 0.0;
      P.MJ[4 * sa + sb] += wj; P.MJ[4 * sb + sa] += wj;
      P.MK[4 * sa + sb] += wk; P.MK[4 * sb + sa] += wk;
      if (wk != 0.0 && as[ua] != 0.0 && as[ub] != 0.0) {
        const int na = slot(2 * ua + 1), nb = slot(2 * ub + 1);
        P.MK[4 * na + nb] += wk; P.MK[4 * nb + na] += wk;
      }
    }
    {
      const int rc_l = launch_classes(ctx, P, 0, d_E, gi == 0, st, stats ? &pool : nullptr, evs, ev_cls, launches);
      if (rc_l) return rc_l;
    }
  }
  CK(cudaGetLastError());
  if (d_E) {
    CK(cudaMemcpyAsync(E_host, d_E, sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
  }
  if (stats) {
    cudaEventRecord(ev2, st);
    CK(cudaStreamSynchronize(st));
    std::vector<unsigned long long> cnt(nw * 3 + 3);
    CK(cudaMemcpy(cnt.data(), ctx->d_counters, sizeof(unsigned long long) * cnt.size(), cudaMemcpyDeviceToHost));
    std::memset(stats, 0, sizeof(*stats));
    stats->pairs_total = ctx->pairs_total; stats->pairs_kept = ctx->pairs_kept;
    for (size_t w = 0; w < nw; ++w) {
      stats->quartets_visited += (int64_t)cnt[3 * w]; stats->quartets_computed += (int64_t)cnt[3 * w + 1];
      stats->prim_quartets += (int64_t)cnt[3 * w + 2];
      stats->quartets_by_class[ctx->work[w].cls] += (int64_t)cnt[3 * w + 1];
      stats->prim_quartets_by_class[ctx->work[w].cls] += (int64_t)cnt[3 * w + 2];
    }
    for (size_t e = 0; e < ev_cls.size(); ++e) {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, evs[2 * e], evs[2 * e + 1]);
      stats->ms_by_class[ev_cls[e]] += ms;
    }
    cudaEventElapsedTime(&stats->ms_prepare, ev0, ev1);
    cudaEventElapsedTime(&stats->ms_total, ev0, ev2);
    stats->launches = launches + aux_launches;
    stats->groups = (int32_t)groups.size();
  }
  return TDG_OK;
}

extern "C" int tdg_gradient(tdg_ctx* ctx, int npair, const double* const* A, const double* const* B, int matrices_on_device,
                            const double* wJ, const double* wK, double cJ, double cK, double cLR, double omega,
                            void* stream, double* grad, int grad_on_device, tdg_stats* stats) {
  if (!ctx) return TDG_EINVAL;
  if (!A || !B || !wJ || !wK || !grad || npair <= 0 || npair > TDG_MAXP) return TDG_EINVAL;
  for (int k = 0; k < npair; ++k) if (!A[k] || !B[k]) return TDG_EINVAL;
  if (cLR != 0.0 && !(omega > 0.0)) return TDG_EINVAL;
  if (!ctx->planned) return TDG_ENOTPLANNED;
  cudaSetDevice(ctx->device);
  cudaStream_t st = (cudaStream_t)stream;
  int rc = run_contraction(ctx, npair, A, B, matrices_on_device, wJ, wK, cJ, cK, cLR, omega, st, stats);
  if (rc) return rc;
  const size_t gb = sizeof(double) * 3 * ctx->natom;
  if (grad_on_device) CK(cudaMemcpyAsync(grad, ctx->d_grad, gb, cudaMemcpyDeviceToDevice, st));
  else { CK(cudaMemcpyAsync(grad, ctx->d_grad, gb, cudaMemcpyDeviceToHost, st)); CK(cudaStreamSynchronize(st)); }
  return TDG_OK;
}

extern "C" int tdg_energy(tdg_ctx* ctx, int npair, const double* const* A, const double* const* B, int matrices_on_device,
                          const double* wJ, const double* wK, double cJ, double cK, double cLR, double omega,
                          void* stream, double* E_host) {
  if (!ctx) return TDG_EINVAL;
  if (!A || !B || !wJ || !wK || !E_host || npair <= 0 || npair > TDG_MAXP) return TDG_EINVAL;
  for (int k = 0; k < npair; ++k) if (!A[k] || !B[k]) return TDG_EINVAL;
  if (cLR != 0.0 && !(omega > 0.0)) return TDG_EINVAL;
  if (!ctx->planned) return TDG_ENOTPLANNED;
  cudaSetDevice(ctx->device);
  return run_contraction(ctx, npair, A, B, matrices_on_device, wJ, wK, cJ, cK, cLR, omega, (cudaStream_t)stream, nullptr, E_host);
}

// ---- NEXT-1: Fock-type (J/K) build (eq 19, eqs 33-34; kernels in tdg_fock.cuh) ----
extern "C" int tdg_fock(tdg_ctx* ctx, int nmat, const double* const* B, int matrices_on_device, const double* wJ, const double* wK,
                        const double* wKT, double cK, double cLR, double omega, void* stream, double* const* F, int F_on_device,
                        tdg_stats* stats) {
  if (!ctx) return TDG_EINVAL;
  if (!B || !F || !wJ || !wK || !wKT || nmat <= 0 || nmat > TDG_MAXP) return TDG_EINVAL;
  for (int k = 0; k < nmat; ++k) if (!B[k] || !F[k]) return TDG_EINVAL;
  if (cLR != 0.0 && !(omega > 0.0)) return TDG_EINVAL;
  if (!ctx->planned) return TDG_ENOTPLANNED;
  cudaSetDevice(ctx->device);
  cudaStream_t st = (cudaStream_t)stream;
  const int n = ctx->nbf;
  const size_t mbytes = sizeof(double) * (size_t)n * n;
  std::fill(ctx->scratch_used.begin(), ctx->scratch_used.end(), false);
  EventPool pool;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr, ev2 = nullptr;
  if (stats) { ev0 = pool.get(); ev1 = pool.get(); ev2 = pool.get(); if (!ev0 || !ev1 || !ev2) return TDG_ECUDA; cudaEventRecord(ev0, st); }
  std::vector<const double*> bdev(nmat);
  std::vector<double*> fdev(nmat);
  for (int k = 0; k < nmat; ++k) {
    const int rc_in = to_device_cart(ctx, B[k], matrices_on_device, st, &bdev[k]);
    if (rc_in) return rc_in;
    fdev[k] = F[k];
    if (!F_on_device || ctx->any_sph) {   // Cartesian result buffer (transformed / copied out at the end)
      fdev[k] = (double*)scratch_get(ctx, mbytes);
      if (!fdev[k]) { ctx->err = "device allocation of an output matrix failed"; return TDG_ENOMEM; }
    }
    CK(cudaMemsetAsync(fdev[k], 0, mbytes, st));
  }
  const bool useK = (cK != 0.0 || cLR != 0.0);
  // which inputs are nonsymmetric (only matters where wK != wKT: the exchange density wK B + wKT B^T is then nonsymmetric)
  double as[TDG_MAXP] = {0};
  bool need_as = false;
  for (int k = 0; k < nmat; ++k) need_as = need_as || (useK && wK[k] != wKT[k]);
  if (need_as) {
    double* d_as = (double*)scratch_get(ctx, 256);
    if (!d_as) return TDG_ENOMEM;
    CK(cudaMemsetAsync(d_as, 0, 256, st));
    for (int k = 0; k < nmat; ++k) CK(tdg_launch_asym(bdev[k], n, d_as + k, st));
    CK(cudaMemcpyAsync(as, d_as, sizeof(double) * nmat, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
  }
  // canonical slots: S_k = (B_k + B_k^T)/2 carries J (weight 2 wJ) and the symmetric part of the exchange density (wK + wKT);
  // N_k = (B_k - B_k^T)/2 carries the antisymmetric part (wK - wKT) and is finished with F -= G^T
  struct Slot { int mat, kind; double jw, kw; };
  std::vector<Slot> slots;
  double CJ = 0.0, CKs = 0.0;
  for (int k = 0; k < nmat; ++k) {
    CJ = std::max(CJ, std::fabs(wJ[k])); CKs = std::max(CKs, std::fabs(wK[k]) + std::fabs(wKT[k]));
    const double ks = useK ? wK[k] + wKT[k] : 0.0, kn = useK ? wK[k] - wKT[k] : 0.0;
    if (wJ[k] != 0.0 || ks != 0.0) slots.push_back(Slot{k, 0, 2.0 * wJ[k], ks});
    if (kn != 0.0 && as[k] != 0.0) slots.push_back(Slot{k, 1, 0.0, kn});
  }
  CKs *= std::fabs(cK) + std::fabs(cLR);
  KParams P{};
  P.CJ = CJ; P.CK = CKs; P.wmode = 1;
  P.tau = ctx->opt.tau; P.density_weighted = (ctx->opt.tau > 0.0) ? ctx->opt.density_weighted : 0;
  P.nshell = ctx->nshell; P.sample_mod = ctx->opt.sample_mod; P.sample_seed = ctx->opt.sample_seed;
  P.nbf = n; P.cK = cK; P.cLR = cLR; P.omega = omega; P.omega2 = omega * omega; P.use_lr = (cLR != 0.0) ? 1 : 0;
  P.rys_tab = ctx->d_rys;
  int aux_launches = 0;
  if (P.density_weighted) {
    if (!ctx->d_dmax) CK(cudaMalloc(&ctx->d_dmax, sizeof(double) * (size_t)ctx->nshell * ctx->nshell));
    MatList ml{};
    ml.n = nmat;
    for (int i = 0; i < nmat; ++i) ml.m[i] = bdev[i];
    CK(tdg_launch_dmax(ml, n, ctx->d_shells, ctx->nshell, ctx->d_dmax, st));
    P.dmax = ctx->d_dmax;
    aux_launches += 2;
  }
  double* pk = (double*)scratch_get(ctx, 4 * mbytes);
  double* G = (double*)scratch_get(ctx, 4 * mbytes + 8);   // (+8: a size distinct from pk's, the scratch cache keys on bytes)
  if (!pk || !G) { ctx->err = "device allocation of the packed / accumulator arrays failed"; return TDG_ENOMEM; }
  P.pk = pk; P.grad = G;
  const size_t nw = ctx->work.size();
  CK(cudaMemsetAsync(ctx->d_counters, 0, sizeof(unsigned long long) * (nw * 3 + 3), st));
  if (stats) cudaEventRecord(ev1, st);
  int launches = 0;
  std::vector<cudaEvent_t> evs;
  std::vector<int> ev_cls;
  const int npass = (int)((slots.size() + 3) / 4);
  for (int pass = 0; pass < npass; ++pass) {
    PackSrc ps{};
    for (int t = 0; t < 4; ++t) { P.MJ[t] = 0.0; P.MK[t] = 0.0; }
    const int s0 = pass * 4, s1 = std::min((int)slots.size(), s0 + 4);
    for (int s = s0; s < s1; ++s) {
      ps.src[s - s0] = bdev[slots[s].mat]; ps.kind[s - s0] = slots[s].kind;
      P.MJ[s - s0] = slots[s].jw; P.MK[s - s0] = slots[s].kw;
    }
    CK(tdg_launch_pack(ps, n, ctx->d_bf2sh, ctx->d_shells, pk, st));
    CK(cudaMemsetAsync(G, 0, 4 * mbytes, st));
    aux_launches += 2;
    {
      const int rc_l = launch_classes(ctx, P, TDG_FOCK_ROLE_BASE, nullptr, pass == 0, st, stats ? &pool : nullptr, evs, ev_cls, launches);
      if (rc_l) return rc_l;
    }
    for (int s = s0; s < s1; ++s) {
      CK(tdg_launch_fock_finalize(G + (size_t)(s - s0) * n * n, n, slots[s].kind == 0 ? 1.0 : -1.0, fdev[slots[s].mat], st));
      ++aux_launches;
    }
  }
  CK(cudaGetLastError());
  {
    const size_t nin = (size_t)ctx->nbf_in, obytes = sizeof(double) * nin * nin;
    for (int k = 0; k < nmat; ++k) {
      const double* res = fdev[k];
      if (ctx->any_sph) {   // F_sph = C F_cart C^T
        double* o = F_on_device ? F[k] : (double*)scratch_get(ctx, obytes);
        if (!o) { ctx->err = "device allocation of an output matrix failed"; return TDG_ENOMEM; }
        CK(tdg_launch_sph_transform(fdev[k], o, (int)nin, n, 1, ctx->d_in2sh, ctx->d_shells, ctx->d_inoff, ctx->d_sph, st));
        res = o;
      }
      if (!F_on_device) CK(cudaMemcpyAsync(F[k], res, obytes, cudaMemcpyDeviceToHost, st));
    }
    if (!F_on_device) CK(cudaStreamSynchronize(st));
  }
  if (stats) {
    cudaEventRecord(ev2, st);
    CK(cudaStreamSynchronize(st));
    std::vector<unsigned long long> cnt(nw * 3 + 3);
    CK(cudaMemcpy(cnt.data(), ctx->d_counters, sizeof(unsigned long long) * cnt.size(), cudaMemcpyDeviceToHost));
    std::memset(stats, 0, sizeof(*stats));
    stats->pairs_total = ctx->pairs_total; stats->pairs_kept = ctx->pairs_kept;
    for (size_t w = 0; w < nw; ++w) {
      stats->quartets_visited += (int64_t)cnt[3 * w]; stats->quartets_computed += (int64_t)cnt[3 * w + 1];
      stats->prim_quartets += (int64_t)cnt[3 * w + 2];
      stats->quartets_by_class[ctx->work[w].cls] += (int64_t)cnt[3 * w + 1];
      stats->prim_quartets_by_class[ctx->work[w].cls] += (int64_t)cnt[3 * w + 2];
    }
    for (size_t e = 0; e < ev_cls.size(); ++e) {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, evs[2 * e], evs[2 * e + 1]);
      stats->ms_by_class[ev_cls[e]] += ms;
    }
    cudaEventElapsedTime(&stats->ms_prepare, ev0, ev1);
    cudaEventElapsedTime(&stats->ms_total, ev0, ev2);
    stats->launches = launches + aux_launches;
    stats->groups = npass;
  }
  return TDG_OK;
}

// ---- NEXT-4: one-electron terms of the gradient (eq 7 terms 1-3; kernels in tdg_onee.cu) ----
extern "C" int tdg_onee_gradient(tdg_ctx* ctx, const double* Z, const double* Pm, const double* Wm, int matrices_on_device, void* stream,
                                 double* grad, int grad_on_device, float* ms) {
  if (!ctx || !Z || !grad) return TDG_EINVAL;
  if (!ctx->planned) return TDG_ENOTPLANNED;
  cudaSetDevice(ctx->device);
  cudaStream_t st = (cudaStream_t)stream;
  std::fill(ctx->scratch_used.begin(), ctx->scratch_used.end(), false);
  EventPool pool;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  if (ms) { ev0 = pool.get(); ev1 = pool.get(); if (!ev0 || !ev1) return TDG_ECUDA; cudaEventRecord(ev0, st); }
  const double *dP = nullptr, *dW = nullptr;
  if (Pm) { const int rc = to_device_cart(ctx, Pm, matrices_on_device, st, &dP); if (rc) return rc; }
  if (Wm) { const int rc = to_device_cart(ctx, Wm, matrices_on_device, st, &dW); if (rc) return rc; }
  double* dZ = (double*)scratch_get(ctx, sizeof(double) * ctx->natom + 16);
  if (!dZ) { ctx->err = "device allocation of the nuclear charges failed"; return TDG_ENOMEM; }
  CK(cudaMemcpyAsync(dZ, Z, sizeof(double) * ctx->natom, cudaMemcpyHostToDevice, st));
  CK(cudaMemsetAsync(ctx->d_grad, 0, sizeof(double) * 3 * ctx->natom, st));
  if (dP || dW)
    for (const Bucket& X : ctx->buckets)
      CK(tdg_launch_onee(X.d_hdr, X.d_prim, X.n, X.npp, X.la, X.lb, ctx->d_xyz, dZ, ctx->natom, dP, dW, ctx->nbf, ctx->d_grad, ctx->d_rys, st));
  CK(tdg_launch_vnuc_grad(ctx->d_xyz, dZ, ctx->natom, ctx->d_grad, st));
  const size_t gb = sizeof(double) * 3 * ctx->natom;
  if (grad_on_device) CK(cudaMemcpyAsync(grad, ctx->d_grad, gb, cudaMemcpyDeviceToDevice, st));
  else CK(cudaMemcpyAsync(grad, ctx->d_grad, gb, cudaMemcpyDeviceToHost, st));
  if (ms) cudaEventRecord(ev1, st);
  CK(cudaStreamSynchronize(st));   // Z (and host matrices) are the caller's host arrays: their uploads finish before the call returns
  if (ms) cudaEventElapsedTime(ms, ev0, ev1);
  return TDG_OK;
}

extern "C" int tdg_rys(tdg_ctx* ctx, int n, int count, const double* T, const double* rho, double omega, double* out) {
  if (!ctx || !T || !rho || !out || n < 1 || n > 7 || count <= 0) return TDG_EINVAL;
  cudaSetDevice(ctx->device);
  DevTemp dT, dr, dout;
  CK(cudaMalloc(&dT.p, sizeof(double) * count)); CK(cudaMalloc(&dr.p, sizeof(double) * count));
  CK(cudaMalloc(&dout.p, sizeof(double) * (size_t)count * 2 * n));
  CK(cudaMemcpy(dT.p, T, sizeof(double) * count, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(dr.p, rho, sizeof(double) * count, cudaMemcpyHostToDevice));
  CK(tdg_launch_rys(n, count, (const double*)dT.p, (const double*)dr.p, omega, ctx->d_rys, (double*)dout.p, 0));
  CK(cudaMemcpy(out, dout.p, sizeof(double) * (size_t)count * 2 * n, cudaMemcpyDeviceToHost));
  return TDG_OK;
}

// Allocation-free variant of tdg_rys (workspace: the file-scope device array of tdg_noalloc.cu; no cudaMalloc / cudaFree here).
extern "C" int tdg_rys_static(tdg_ctx* ctx, int n, int count, const double* T, const double* rho, double omega, void* stream, double* out) {
  if (!ctx || !T || !rho || !out || n < 1 || n > 7 || count <= 0) return TDG_EINVAL;
  if (count > tdg_rys_static_max()) {
    ctx->err = "tdg_rys_static: count " + std::to_string(count) + " exceeds the fixed workspace (TDG_RYS_STATIC_MAX = " +
               std::to_string(tdg_rys_static_max()) + " evaluations per call); split the batch or use tdg_rys";
    return TDG_EINVAL;
  }
  cudaSetDevice(ctx->device);
  unsigned long long nbad = 0;
  CK(tdg_run_rys_static(ctx->device, n, count, T, rho, omega, ctx->d_rys, out, &nbad, (cudaStream_t)stream));
  if (nbad) { ctx->err = "tdg_rys_static: " + std::to_string(nbad) + " argument(s) with T < 0, rho <= 0, NaN or infinity"; return TDG_EINVAL; }
  return TDG_OK;
}

extern "C" int tdg_fp64_peak(tdg_ctx* ctx, double ms, double* tflops) {
  if (!ctx || !tflops) return TDG_EINVAL;
  cudaSetDevice(ctx->device);
  CK(tdg_run_fp64_peak(ms, tflops));
  return TDG_OK;
}
