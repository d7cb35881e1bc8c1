// pwham.cu -- C ABI of libpwham (include/pwham.h): handle setup, workspace carving and the launch sequences of
// apply_h, cheb_filter and gram.  Host code here only builds tables and enqueues kernels; every step of the path
// (scatter, FFTs, V_loc multiply, gather, kinetic, recurrence, projector and Gram contractions) runs in the
// kernels of local_kernels.cu and zgemm.cu.  There is no CPU fallback.
#include "../../include/pwham.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "launch.h"

using namespace pwh;

// NVTX range per stage of the path (the paper isolates its roofline regions the same way);
// header-only NVTX v3: a no-op unless a profiler injects itself.
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};

namespace pwh {
static std::atomic<int64_t> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

// Optional per-launch timing (pwh_profile_begin / pwh_profile_end): one cudaEvent pair around every kernel launch,
// recorded on the launching stream.  Off by default; the hot path then pays one relaxed atomic load per launch.
struct ProfRec { int stage; cudaEvent_t e0, e1; };
static std::atomic<bool> g_prof_on{false};
static std::mutex g_prof_mu;
static std::vector<ProfRec> g_prof;
static std::vector<cudaEvent_t> g_prof_pool;

static cudaEvent_t prof_event() {
  cudaEvent_t e = nullptr;
  if (!g_prof_pool.empty()) { e = g_prof_pool.back(); g_prof_pool.pop_back(); }
  else cudaEventCreate(&e);
  return e;
}
ScopedLaunch::ScopedLaunch(int stage, cudaStream_t st) : st_(st), idx_(-1) {
  count_launch();
  if (!g_prof_on.load(std::memory_order_relaxed)) return;
  std::lock_guard<std::mutex> lk(g_prof_mu);
  ProfRec r{stage, prof_event(), prof_event()};
  cudaEventRecord(r.e0, st_);
  idx_ = (int64_t)g_prof.size();
  g_prof.push_back(r);
}
ScopedLaunch::~ScopedLaunch() {
  if (idx_ < 0) return;
  std::lock_guard<std::mutex> lk(g_prof_mu);
  cudaEventRecord(g_prof[(size_t)idx_].e1, st_);
}
cudaError_t set_max_dyn_smem(const void* func) {
  int dev = 0, smem_max = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (e != cudaSuccess) return e;
  cudaFuncAttributes fa;
  e = cudaFuncGetAttributes(&fa, func);
  if (e != cudaSuccess) return e;
  // static + dynamic shared memory together must stay within the opt-in maximum
  return cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max - (int)fa.sharedSizeBytes);
}
}  // namespace pwh

static thread_local std::string g_err;

static int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}

namespace pwh {
int api_fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}
}  // namespace pwh

#define CUDA_TRY(expr)                                                                        \
  do {                                                                                        \
    cudaError_t e__ = (expr);                                                                 \
    if (e__ != cudaSuccess)                                                                   \
      return fail(e__ == cudaErrorMemoryAllocation ? PWH_ENOMEM : PWH_ECUDA, "%s: %s", #expr, \
                  cudaGetErrorString(e__));                                                   \
  } while (0)

struct pwh_ham {
  int64_t npw = 0, nproj = 0;
  int n1 = 0, n2 = 0, n3 = 0;
  LocalPlan lp;
  FastPlan fp;
  bool fast = false;
  V2Plan vp;
  bool v2 = false;
  ZPlan zp;
  bool zw = false;
  const c128* proj = nullptr;
  int64_t ldp = 0;
  ProjMaps pmaps;
  double* dij = nullptr;
  int band_group = 1;
  const int* dnat[3] = {nullptr, nullptr, nullptr};   // generic stage plan: position -> natural index per axis
  // PAW-style generalised problem (pwh_ham_set_paw): per-atom dense D^R / Q^R blocks and K of S^-1 = I - P K P^H
  bool paw = false;
  int* blk_of = nullptr;         // [nproj] block (atom) of each projector
  int* blk_lo = nullptr;         // [nblk + 1] first projector of each block
  int64_t* boff = nullptr;       // [nblk] element offset of each packed block
  c128* dblk = nullptr;          // packed column-major blocks D^R
  c128* qblk = nullptr;          // packed column-major blocks Q^R
  c128* kmat = nullptr;          // nproj x nproj, K
  std::vector<void*> allocs;
  // staging of the *_host entry points
  void* st_psi = nullptr;
  void* st_hpsi = nullptr;
  void* st_g = nullptr;
  void* st_ws = nullptr;
  size_t st_psi_bytes = 0, st_hpsi_bytes = 0, st_g_bytes = 0, st_ws_bytes = 0;
  // copy streams and events of the pipelined host entry points
  cudaStream_t cs_in = nullptr, cs_out = nullptr;
  std::vector<cudaEvent_t> evs;
  // the band groups of the local stage alternate between two internal streams (each with its own column buffer), so that
  // the partial last wave of one group's kernels is filled by the other group's (lways = 1: one stream, in order)
  int lways = 1;
  int lbufs = 1;                 // column buffers in the workspace layout (fixed at setup: the layout never changes)
  cudaStream_t ls[2] = {nullptr, nullptr};
  cudaEvent_t lev_fork = nullptr, lev_join[2] = {nullptr, nullptr};
  // one or two streams?  Measured, not guessed (profiles/r02h): two streams win where the z kernels are a large part of the
  // stage (cfg 5), one stream where the plane kernel dominates (cfg 3, 4) -- by about 1 % of the step either way.  The first
  // four multi-group H applications of a handle alternate between the two and are bracketed by events on the caller's
  // stream; a later call reads the four times back with cudaEventQuery (no host synchronisation anywhere) and fixes the
  // choice.  The results do not depend on it (every band runs through the same kernels).
  bool ltune = false;            // still deciding
  int ltune_calls = 0;
  int64_t ltune_nband = 0;
  cudaEvent_t ltune_ev[4][2] = {};
};

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ---------------------------------------------------------------------------------------------------------------
// setup helpers
// ---------------------------------------------------------------------------------------------------------------
static bool factor_235(int n, int& e2, int& e3, int& e5) {
  e2 = e3 = e5 = 0;
  while (n % 2 == 0) { n /= 2; ++e2; }
  while (n % 3 == 0) { n /= 3; ++e3; }
  while (n % 5 == 0) { n /= 5; ++e5; }
  return n == 1;
}

// radix schedule: 8s, 4s, 5s, 3s, then a lone 2 (8*2 is re-split into 4*4)
static bool make_axis_plan(int n, AxisPlan& pl, std::vector<c128>& tw, std::vector<int>& nat) {
  int e2, e3, e5;
  if (n < 2 || !factor_235(n, e2, e3, e5)) return false;
  std::vector<int> rad;
  int n8 = e2 / 3, rem = e2 % 3, n4 = 0, n2 = 0;
  if (rem == 1) {
    if (n8 >= 1) { --n8; n4 += 2; } else n2 = 1;
  } else if (rem == 2) n4 += 1;
  for (int i = 0; i < n8; ++i) rad.push_back(8);
  for (int i = 0; i < n4; ++i) rad.push_back(4);
  for (int i = 0; i < e5; ++i) rad.push_back(5);
  for (int i = 0; i < e3; ++i) rad.push_back(3);
  for (int i = 0; i < n2; ++i) rad.push_back(2);
  if ((int)rad.size() > PWH_MAX_STAGES) return false;
  memset(&pl, 0, sizeof(pl));
  pl.n = n;
  pl.nstages = (int)rad.size();
  tw.clear();
  int B = n;
  const long double PI = 3.14159265358979323846264338327950288L;
  for (int s = 0; s < pl.nstages; ++s) {
    const int r = rad[s], m = B / r;
    pl.radix[s] = r;
    pl.m[s] = m;
    pl.div_m[s] = make_fastdiv((uint32_t)m);
    pl.tw_off[s] = (int)tw.size();
    if (m > 1) {
      for (int k = 1; k < r; ++k)
        for (int n2i = 0; n2i < m; ++n2i) {
          const long t = ((long)n2i * k) % B;
          const long double ang = 2.0L * PI * (long double)t / (long double)B;
          tw.push_back(cmake((double)cosl(ang), (double)sinl(ang)));
        }
    }
    B = m;
  }
  pl.tw_len = (int)tw.size();
  // position -> natural index of the digit-permuted order
  nat.assign(n, 0);
  std::vector<int> cur(1, 0);
  int size = 1;
  for (int s = pl.nstages - 1; s >= 0; --s) {
    const int r = rad[s];
    std::vector<int> next((size_t)size * r);
    for (int k1 = 0; k1 < r; ++k1)
      for (int p = 0; p < size; ++p) next[(size_t)k1 * size + p] = k1 + r * cur[p];
    cur.swap(next);
    size *= r;
  }
  nat = cur;
  return true;
}

// n = r1 * r2 with r1 in {1..6,8,9,10,12,15,16}, r2 in {1..6,8,9,10,12}, r1 >= r2, |r1 - r2| minimal; n <= 16 -> r2 = 1
static bool factor_two_pass(int n, int& r1, int& r2) {
  static const int S1[] = {1, 2, 3, 4, 5, 6, 8, 9, 10, 12, 15, 16};
  static const int S2[] = {1, 2, 3, 4, 5, 6, 8, 9, 10, 12};
  auto in = [](const int* s, int len, int v) { for (int i = 0; i < len; ++i) if (s[i] == v) return true; return false; };
  if (n <= 16 && in(S1, 12, n)) { r1 = n; r2 = 1; return true; }
  int best = -1;
  for (int b : S2) {
    if (b < 2 || n % b) continue;
    const int a = n / b;
    if (a < b || !in(S1, 12, a)) continue;
    if (best < 0 || a - b < best) { best = a - b; r1 = a; r2 = b; }
  }
  return best >= 0;
}

// V_loc/F in slot order, y-slot fastest: out[(zs*n1 + xs)*n2 + ys] = v[px(xs) + n1*(py(ys) + n2*pz(zs))] / F,
// p(s) = s / r2 + r1 * (s % r2)
__global__ void k_slot_vloc(int n1, int n2, int n3, int r1x, int r2x, int r1y, int r2y, int r1z, int r2z,
                            const double* __restrict__ v, double inv_f, double* __restrict__ out) {
  const int64_t total = (int64_t)n1 * n2 * n3;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int ys = (int)(i % n2);
    const int xs = (int)((i / n2) % n1);
    const int zs = (int)(i / ((int64_t)n1 * n2));
    const int x = xs / r2x + r1x * (xs % r2x), y = ys / r2y + r1y * (ys % r2y), z = zs / r2z + r1z * (zs % r2z);
    out[i] = v[x + (int64_t)n1 * (y + (int64_t)n2 * z)] * inv_f;
  }
}

__global__ void k_permute_vloc(int n1, int n2, int n3, const double* __restrict__ v, const int* __restrict__ natx,
                               const int* __restrict__ naty, const int* __restrict__ natz, double inv_f,
                               double* __restrict__ out) {
  const int64_t total = (int64_t)n1 * n2 * n3;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int px = (int)(i % n1);
    const int py = (int)((i / n1) % n2);
    const int pz = (int)(i / ((int64_t)n1 * n2));
    out[i] = v[natx[px] + (int64_t)n1 * (naty[py] + (int64_t)n2 * natz[pz])] * inv_f;
  }
}

template <typename T>
static int upload(pwh_ham* h, const std::vector<T>& v, const T** out, cudaStream_t st) {
  void* d = nullptr;
  const size_t bytes = std::max<size_t>(v.size() * sizeof(T), 16);
  CUDA_TRY(cudaMalloc(&d, bytes));
  h->allocs.push_back(d);
  if (!v.empty()) CUDA_TRY(cudaMemcpyAsync(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st));
  *out = reinterpret_cast<const T*>(d);
  return PWH_OK;
}

// Kernel-family switches for the tests (documented in include/pwham.h); sampled by pwh_ham_setup only, never on a launch path.
static bool env_on(const char* name) {
  const char* e = getenv(name);
  return e && e[0] == '1';
}

static int wrapi(int v, int n) {
  int r = v % n;
  return r < 0 ? r + n : r;
}

extern "C" int pwh_ham_destroy(pwh_ham* h) {
  if (!h) return PWH_OK;
  for (void* p : h->allocs) cudaFree(p);
  if (h->st_psi) cudaFree(h->st_psi);
  if (h->st_hpsi) cudaFree(h->st_hpsi);
  if (h->st_g) cudaFree(h->st_g);
  if (h->st_ws) cudaFree(h->st_ws);
  if (h->cs_in) cudaStreamDestroy(h->cs_in);
  if (h->cs_out) cudaStreamDestroy(h->cs_out);
  for (cudaEvent_t e : h->evs) cudaEventDestroy(e);
  for (int i = 0; i < 2; ++i) {
    if (h->ls[i]) cudaStreamDestroy(h->ls[i]);
    if (h->lev_join[i]) cudaEventDestroy(h->lev_join[i]);
  }
  if (h->lev_fork) cudaEventDestroy(h->lev_fork);
  for (auto& pr : h->ltune_ev)
    for (cudaEvent_t e : pr)
      if (e) cudaEventDestroy(e);
  delete h;
  return PWH_OK;
}

static int setup_impl(pwh_ham* h, const double lattice[9], const double kpt[3], const int32_t dims[3], int64_t npw,
                      const int32_t* gvec, const double* vloc, int64_t nproj, const pwh_c128* proj, int64_t ldp,
                      const double* dij, cudaStream_t st) {
  const int n1 = dims[0], n2 = dims[1], n3 = dims[2];
  h->npw = npw;
  h->nproj = nproj;
  h->n1 = n1; h->n2 = n2; h->n3 = n3;
  h->proj = reinterpret_cast<const c128*>(proj);
  h->ldp = ldp;
  LocalPlan& lp = h->lp;
  memset(&lp, 0, sizeof(lp));
  lp.n1 = n1; lp.n2 = n2; lp.n3 = n3;

  // FFT plans: register-resident two-pass plan when every axis factors as r1 * r2, otherwise the generic
  // radix-2/3/4/5/8 shared-memory stages (PWH_FORCE_GENERIC_FFT=1 forces the latter; used by the tests)
  FastPlan& fp = h->fp;
  memset(&fp, 0, sizeof(fp));
  {
    bool ok = !env_on("PWH_FORCE_GENERIC_FFT");
    for (int ax = 0; ax < 3 && ok; ++ax) ok = factor_two_pass(dims[ax], fp.r1[ax], fp.r2[ax]);
    h->fast = ok;
  }
  zgemm_set_no_tma(env_on("PWH_ZGEMM_NO_TMA"));
  std::vector<c128> tw[3];
  std::vector<int> nat[3];
  for (int ax = 0; ax < 3; ++ax)
    if (!make_axis_plan(dims[ax], lp.ax[ax], tw[ax], nat[ax]))
      return fail(PWH_EUNSUPPORTED, "fft_dims[%d] = %d: only sizes >= 2 with prime factors 2, 3, 5 are supported", ax,
                  dims[ax]);
  if (n1 > 4096 || n2 > 4096 || n3 > 4096) return fail(PWH_EUNSUPPORTED, "fft_dims larger than 4096 not supported");

  // G vectors to the host (once), validation
  std::vector<int32_t> g((size_t)npw * 3);
  CUDA_TRY(cudaMemcpyAsync(g.data(), gvec, g.size() * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  const size_t F = (size_t)n1 * n2 * n3;
  {
    std::vector<bool> seen(F, false);
    for (int64_t i = 0; i < npw; ++i) {
      const size_t idx = wrapi(g[3 * i], n1) + (size_t)n1 * (wrapi(g[3 * i + 1], n2) + (size_t)n2 * wrapi(g[3 * i + 2], n3));
      if (seen[idx]) return fail(PWH_EINVAL, "gvec: plane wave %lld collides with another one in the FFT box", (long long)i);
      seen[idx] = true;
    }
  }

  // kinetic diagonal 1/2 |B (k + n)|^2, B = 2 pi (A^-1)^T
  {
    const double* a = lattice;
    const double det = a[0] * (a[4] * a[8] - a[5] * a[7]) - a[1] * (a[3] * a[8] - a[5] * a[6]) +
                       a[2] * (a[3] * a[7] - a[4] * a[6]);
    if (!(std::fabs(det) > 0.0)) return fail(PWH_EINVAL, "lattice is singular");
    const double tp = 6.283185307179586476925286766559 / det;
    const double b1[3] = {tp * (a[4] * a[8] - a[5] * a[7]), tp * (a[5] * a[6] - a[3] * a[8]), tp * (a[3] * a[7] - a[4] * a[6])};
    const double b2[3] = {tp * (a[7] * a[2] - a[8] * a[1]), tp * (a[8] * a[0] - a[6] * a[2]), tp * (a[6] * a[1] - a[7] * a[0])};
    const double b3[3] = {tp * (a[1] * a[5] - a[2] * a[4]), tp * (a[2] * a[3] - a[0] * a[5]), tp * (a[0] * a[4] - a[1] * a[3])};
    std::vector<double> kin((size_t)npw);
    for (int64_t i = 0; i < npw; ++i) {
      const double c0 = kpt[0] + g[3 * i], c1 = kpt[1] + g[3 * i + 1], c2 = kpt[2] + g[3 * i + 2];
      double q2 = 0.0;
      for (int d = 0; d < 3; ++d) {
        const double q = c0 * b1[d] + c1 * b2[d] + c2 * b3[d];
        q2 += q * q;
      }
      kin[i] = 0.5 * q2;
    }
    int rc = upload(h, kin, &lp.kin, st);
    if (rc) return rc;
  }

  // z-columns touched by the sphere, ordered by the signed (gy, gx) of their first member
  struct Col { int xw, yw, gx, gy; };
  std::vector<int> col_of_xy((size_t)n1 * n2, -1);
  std::vector<Col> cols;
  for (int64_t i = 0; i < npw; ++i) {
    const int xw = wrapi(g[3 * i], n1), yw = wrapi(g[3 * i + 1], n2);
    int& c = col_of_xy[(size_t)yw * n1 + xw];
    if (c < 0) {
      c = (int)cols.size();
      cols.push_back({xw, yw, g[3 * i], g[3 * i + 1]});
    }
  }
  std::vector<int> order(cols.size());
  for (size_t i = 0; i < order.size(); ++i) order[i] = (int)i;
  std::sort(order.begin(), order.end(), [&](int a_, int b_) {
    const Col &A = cols[a_], &B = cols[b_];
    return A.gy != B.gy ? A.gy < B.gy : (A.gx != B.gx ? A.gx < B.gx : a_ < b_);
  });
  std::vector<int> rank(cols.size());
  for (size_t r = 0; r < order.size(); ++r) rank[order[r]] = (int)r;
  const int ncols = (int)cols.size();

  // x-lines touched, ordered by signed gx
  std::vector<int> xl_gx(n1, INT32_MAX);
  for (const Col& c : cols) xl_gx[c.xw] = std::min(xl_gx[c.xw], c.gx);
  std::vector<int> xs;
  for (int x = 0; x < n1; ++x)
    if (xl_gx[x] != INT32_MAX) xs.push_back(x);
  std::sort(xs.begin(), xs.end(), [&](int a_, int b_) { return xl_gx[a_] != xl_gx[b_] ? xl_gx[a_] < xl_gx[b_] : a_ < b_; });
  const int nxl = (int)xs.size();
  std::vector<short> xl_of_x(n1, -1), x_of_xl(nxl);
  for (int i = 0; i < nxl; ++i) { xl_of_x[xs[i]] = (short)i; x_of_xl[i] = (short)xs[i]; }

  lp.ncols = ncols;
  lp.nxl = nxl;
  lp.colgrp = h->fast ? 32 : 16;
  lp.ngrp = (ncols + 2 + lp.colgrp - 1) / lp.colgrp;   // at least two padding columns (kv2_plane: a zero one and a dump)
  lp.ncols_pad = lp.ngrp * lp.colgrp;
  lp.zstride = n3 | 1;
  lp.ystride = n2 | 1;
  lp.xstride = n1 | 1;
  int xb = 1;
  for (int d = 1; d <= 32 && d <= n2; ++d)
    if (n2 % d == 0) xb = d;
  lp.xbatch = xb;
  lp.div_colgrp = make_fastdiv(lp.colgrp);
  lp.div_nxl = make_fastdiv(nxl);
  lp.div_xbatch = make_fastdiv(xb);
  lp.div_n1 = make_fastdiv(n1);
  lp.div_ncols_pad = make_fastdiv(lp.ncols_pad);

  std::vector<int> col_hp(lp.ncols_pad, -1);
  for (size_t i = 0; i < cols.size(); ++i) col_hp[rank[i]] = xl_of_x[cols[i].xw] * lp.ystride + cols[i].yw;

  // sphere entries sorted by (column group, plane-wave index)
  std::vector<int> ent_grp((size_t)npw), ent_off((size_t)npw), perm((size_t)npw);
  for (int64_t i = 0; i < npw; ++i) {
    const int xw = wrapi(g[3 * i], n1), yw = wrapi(g[3 * i + 1], n2), zw = wrapi(g[3 * i + 2], n3);
    const int c = rank[col_of_xy[(size_t)yw * n1 + xw]];
    ent_grp[i] = c / lp.colgrp;
    ent_off[i] = (c % lp.colgrp) * lp.zstride + zw;
    perm[i] = (int)i;
  }
  std::stable_sort(perm.begin(), perm.end(), [&](int a_, int b_) { return ent_grp[a_] < ent_grp[b_]; });
  std::vector<int> grp_ptr(lp.ngrp + 1, 0), ent_pw_s((size_t)npw), ent_off_s((size_t)npw);
  for (int64_t e = 0; e < npw; ++e) {
    ent_pw_s[e] = perm[e];
    ent_off_s[e] = ent_off[perm[e]];
    grp_ptr[ent_grp[perm[e]] + 1]++;
  }
  for (int gi = 0; gi < lp.ngrp; ++gi) grp_ptr[gi + 1] += grp_ptr[gi];

  int rc;
  if ((rc = upload(h, grp_ptr, &lp.grp_ptr, st))) return rc;
  if ((rc = upload(h, ent_pw_s, &lp.ent_pw, st))) return rc;
  if ((rc = upload(h, ent_off_s, &lp.ent_off, st))) return rc;
  if ((rc = upload(h, col_hp, &lp.col_hp, st))) return rc;
  if ((rc = upload(h, xl_of_x, &lp.xl_of_x, st))) return rc;
  if ((rc = upload(h, x_of_xl, &lp.x_of_xl, st))) return rc;
  for (int ax = 0; ax < 3; ++ax)
    if ((rc = upload(h, tw[ax], &lp.tw[ax], st))) return rc;
  {
    std::vector<AxisPlan> plans(lp.ax, lp.ax + 3);
    if ((rc = upload(h, plans, &lp.axp, st))) return rc;
  }

  int dev = 0, smem_max = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));

  if (h->fast) {
    fp.n1 = n1; fp.n2 = n2; fp.n3 = n3;
    fp.ncols = ncols; fp.ncols_pad = lp.ncols_pad; fp.nxl = nxl;
    fp.colgrp = lp.colgrp; fp.ngrp = lp.ngrp;
    fp.zstride = lp.zstride; fp.ystride = lp.ystride;
    fp.grp_ptr = lp.grp_ptr; fp.ent_pw = lp.ent_pw; fp.ent_off = lp.ent_off; fp.col_hp = lp.col_hp;
    fp.xl_of_x = lp.xl_of_x; fp.kin = lp.kin;
    fp.div_colgrp = lp.div_colgrp; fp.div_nxl = lp.div_nxl;
    // full twiddle tables exp(+2 pi i t / n)
    const long double PI = 3.14159265358979323846264338327950288L;
    for (int ax = 0; ax < 3; ++ax) {
      std::vector<c128> t((size_t)dims[ax]);
      for (int k = 0; k < dims[ax]; ++k) {
        const long double ang = 2.0L * PI * (long double)k / (long double)dims[ax];
        t[k] = cmake((double)cosl(ang), (double)sinl(ang));
      }
      if ((rc = upload(h, t, &fp.tw[ax], st))) return rc;
    }
    // y-slots per x batch: the largest divisor of n2 that is <= 32 (all of n2 when the x transform is one pass);
    // shrink it until the plane fits in shared memory; prefer two 256-thread CTAs per SM when they fit
    if (fp.r2[0] == 1) { fp.yb = n2; fp.tsize = 0; }
    else {
      int yb = 1;
      for (int d = 1; d <= 32 && d <= n2; ++d) if (n2 % d == 0) yb = d;
      fp.yb = yb; fp.tsize = n1 * yb;
      while (fast_plane_smem(fp) > (size_t)smem_max && fp.yb > 1) {
        int nb = 1;
        for (int d = 1; d < fp.yb; ++d) if (n2 % d == 0) nb = d;
        fp.yb = nb; fp.tsize = n1 * nb;
      }
    }
    fp.div_yb = make_fastdiv(fp.yb);
    if (fast_plane_smem(fp) > (size_t)smem_max || fast_zkernel_smem(fp) > (size_t)smem_max) h->fast = false;
  }
  // size-specialised plane kernel (local_v2.cu): needs the register-resident z kernels, a box side it is instantiated
  // for, x-lines contiguous modulo n1 and every y-row of the disc a contiguous run of x-lines (true for any convex cutoff
  // sphere; otherwise the generic-size plane kernel of local_fast.cu serves)
  if (h->fast) {
    bool pre = nxl < 65536 && ncols < (1 << 30);
    for (int i = 0; i < nxl && pre; ++i) pre = x_of_xl[i] == (x_of_xl[0] + i) % n1;
    std::vector<int2> yrow((size_t)n2, make_int2(0, 0));
    int nyl = n2;
    if (pre) {
      std::vector<int> row_gy(n2, INT32_MAX), row_first(n2, 0), row_xlmin(n2, 0), row_cnt(n2, 0);
      for (int r = 0; r < ncols && pre; ++r) {
        const Col& c = cols[order[r]];
        const int xl = xl_of_x[c.xw];
        if (row_cnt[c.yw] == 0) { row_gy[c.yw] = c.gy; row_first[c.yw] = r; row_xlmin[c.yw] = xl; row_cnt[c.yw] = 1; }
        else {
          pre = row_gy[c.yw] == c.gy && r == row_first[c.yw] + row_cnt[c.yw] && xl == row_xlmin[c.yw] + row_cnt[c.yw];
          row_cnt[c.yw]++;
        }
      }
      // rows indexed from the lowest touched one (signed gy): yl = (y - y0) mod n2, so that the disc is a prefix of the axis
      int gy_min = INT32_MAX, gy_max = INT32_MIN;
      for (int y = 0; y < n2; ++y)
        if (row_cnt[y] > 0) { gy_min = std::min(gy_min, row_gy[y]); gy_max = std::max(gy_max, row_gy[y]); }
      nyl = gy_max - gy_min + 1;
      pre = pre && nyl >= 1 && nyl <= n2;
      for (int yl = 0; yl < n2 && pre; ++yl) {
        const int y = wrapi(gy_min + yl, n2);
        yrow[yl] = make_int2(row_first[y] - row_xlmin[y], row_xlmin[y] | (row_cnt[y] << 16));
      }
    }
    const long double PI = 3.14159265358979323846264338327950288L;
    V2Plan& vp = h->vp;
    memset(&vp, 0, sizeof(vp));
    if (pre && !env_on("PWH_NO_V2") && v2_select(vp, n1, n2, nxl, nyl, (size_t)smem_max, env_on("PWH_V2_NO_PRUNE"))) {
      vp.n1 = n1; vp.n2 = n2; vp.n3 = n3; vp.ncols_pad = lp.ncols_pad; vp.nxl = nxl; vp.x0 = x_of_xl[0];
      vp.zcol = ncols;
      vp.div_nxl = lp.div_nxl;
      if ((rc = upload(h, yrow, &vp.yrow, st))) return rc;
      for (int ax = 0; ax < 2; ++ax) {
        const int n = dims[ax], r1 = vp.r1[ax], r2 = vp.r2[ax];
        std::vector<c128> ta((size_t)r2 * (r1 + 1), cmake(0.0, 0.0)), tb((size_t)r1 * (r2 + 1), cmake(0.0, 0.0));
        for (int s_ = 0; s_ < r2; ++s_)
          for (int k1 = 0; k1 < r1; ++k1) {
            const long double ang = 2.0L * PI * (long double)((s_ * k1) % n) / (long double)n;
            const c128 w = cmake((double)cosl(ang), (double)sinl(ang));
            ta[(size_t)s_ * (r1 + 1) + k1] = w;
            tb[(size_t)k1 * (r2 + 1) + s_] = w;
          }
        if ((rc = upload(h, ta, &vp.twA[ax], st))) return rc;
        if ((rc = upload(h, tb, &vp.twB[ax], st))) return rc;
      }
      double* vperm = nullptr;
      CUDA_TRY(cudaMalloc(&vperm, F * sizeof(double)));
      h->allocs.push_back(vperm);
      launch_v2_perm_vloc(vp, fp.r1[2], fp.r2[2], vloc, vperm, st);
      CUDA_TRY(cudaGetLastError());
      vp.vperm = vperm;
      CUDA_TRY(v2_kernels_init(vp));
      h->v2 = true;
    }
  }
  // warp-private z kernels (local_z.cu): table of plane-wave indices in the order their lanes read it
  if (h->fast) {
    ZPlan& zp = h->zp;
    memset(&zp, 0, sizeof(zp));
    zp.n3 = n3; zp.r1 = fp.r1[2]; zp.r2 = fp.r2[2];
    // z-rows counted from the lowest touched z (signed gz): the sphere is a prefix of the axis, nzl rows long
    int gz_min = INT32_MAX, gz_max = INT32_MIN;
    for (int64_t i = 0; i < npw; ++i) { gz_min = std::min(gz_min, (int)g[3 * i + 2]); gz_max = std::max(gz_max, (int)g[3 * i + 2]); }
    const int nzl = gz_max - gz_min + 1;
    zp.lq = zp.r1;
    if (!env_on("PWH_V2_NO_PRUNE") && zp.r2 > 1 && zw_pruned_len(zp.r1) < zp.r1 && nzl <= zw_pruned_len(zp.r1) * zp.r2)
      zp.lq = zw_pruned_len(zp.r1);
    zp.lqp = (zp.lq + 3) / 4 * 4;
    zp.cw = zp.r2 >= 6 ? 4 : (zp.r2 >= 4 ? 8 : (zp.r2 >= 2 ? 16 : 32));
    zp.log2cw = zp.cw == 4 ? 2 : (zp.cw == 8 ? 3 : (zp.cw == 16 ? 4 : 5));
    zp.nq = lp.ncols_pad / zp.cw;
    zp.ncols_pad = lp.ncols_pad;
    // column stride of a warp buffer: cw = 4 lanes x 2 consecutive subs of a quarter-warp need stride == 2 (mod 8),
    // cw >= 8 lanes of a quarter-warp sit on 8 columns and need an odd stride
    int zs = zp.r1 * (zp.r2 + 1);
    if (zp.cw == 4) { while (zs % 8 != 2) ++zs; } else zs |= 1;
    zp.zs = zs;
    zp.tw = fp.tw[2];
    zp.kin = lp.kin;
    if (!env_on("PWH_NO_ZW") && zw_smem(zp) <= (size_t)smem_max && nzl <= n3) {
      std::vector<int> ztab((size_t)zp.nq * zp.r2 * zp.cw * zp.lqp, -1);
      for (int64_t i = 0; i < npw; ++i) {
        const int xw = wrapi(g[3 * i], n1), yw = wrapi(g[3 * i + 1], n2), zl = g[3 * i + 2] - gz_min;
        const int c = rank[col_of_xy[(size_t)yw * n1 + xw]];
        const int quad = c / zp.cw, cl = c % zp.cw, sub = zl % zp.r2, q = zl / zp.r2;
        const size_t nelem = (size_t)zp.r2 * zp.cw, el = (size_t)sub * zp.cw + cl;
        ztab[(((size_t)quad * (zp.lqp / 4) + q / 4) * nelem + el) * 4 + q % 4] = (int)i;
      }
      if ((rc = upload(h, ztab, &zp.ztab, st))) return rc;
      CUDA_TRY(zw_kernels_init(zp));
      h->zw = true;
    }
  }
  if (h->fast) {
    int smem_sm = 0;
    CUDA_TRY(cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev));
    fp.plane_threads = (2 * (fast_plane_smem(fp) + 1024) <= (size_t)smem_sm) ? 256 : 512;
    double* vp = nullptr;
    CUDA_TRY(cudaMalloc(&vp, F * sizeof(double)));
    h->allocs.push_back(vp);
    k_slot_vloc<<<148 * 4, 256, 0, st>>>(n1, n2, n3, fp.r1[0], fp.r2[0], fp.r1[1], fp.r2[1], fp.r1[2], fp.r2[2], vloc,
                                         1.0 / (double)F, vp);
    CUDA_TRY(cudaGetLastError());
    fp.vslot = vp;
    CUDA_TRY(fast_kernels_init(fp));
  } else {
    // generic path: V_loc / F in digit-permuted positions
    const int** dnat = h->dnat;
    for (int ax = 0; ax < 3; ++ax)
      if ((rc = upload(h, nat[ax], &dnat[ax], st))) return rc;
    double* vp = nullptr;
    CUDA_TRY(cudaMalloc(&vp, F * sizeof(double)));
    h->allocs.push_back(vp);
    k_permute_vloc<<<148 * 4, 256, 0, st>>>(n1, n2, n3, vloc, dnat[0], dnat[1], dnat[2], 1.0 / (double)F, vp);
    CUDA_TRY(cudaGetLastError());
    lp.vperm = vp;
    if (plane_smem(lp) > (size_t)smem_max || zkernel_smem(lp) > (size_t)smem_max)
      return fail(PWH_EUNSUPPORTED, "FFT box %dx%dx%d needs %zu bytes of shared memory per plane (limit %d)", n1, n2, n3,
                  plane_smem(lp), smem_max);
    CUDA_TRY(local_kernels_init(lp));
  }

  // D (copied)
  if (nproj > 0) {
    CUDA_TRY(cudaMalloc(&h->dij, nproj * sizeof(double)));
    h->allocs.push_back(h->dij);
    CUDA_TRY(cudaMemcpyAsync(h->dij, dij, nproj * sizeof(double), cudaMemcpyDeviceToDevice, st));
  }

  CUDA_TRY(zgemm_init());
  if (nproj > 0) zgemm_make_proj_maps(h->pmaps, h->proj, npw, nproj, ldp);

  // bands per launch of the local kernels.  The z kernels are latency-bound and want many work items per launch (a group of
  // 4 bands at cfg 5 is 1.19 rounds of the resident warps, i.e. two rounds of which the second is almost empty), the plane
  // kernel's grid of n3 x bands CTAs (one per SM) should fill whole waves of the 148 SMs, and the column buffer of a group
  // (written by one kernel, read by the next) is served from the 126 MB L2 for its most recently written part whatever its
  // size.  Measured (profiles/r02f): the stage gets faster up to about 300 MB of column buffer per group and flat beyond,
  // so among the group sizes with 190 ... 320 MB take the one with the best wave efficiency of the plane kernel.
  const size_t per_band = (size_t)n3 * lp.ncols_pad * sizeof(c128);
  const int64_t slots = 148;                                                            // resident plane CTAs
  const size_t win_hi = 320u << 20, win_lo = 190u << 20;
  const int64_t min_grp = (2 * 148 + n3 - 1) / n3;
  int64_t g_lo = std::max<int64_t>(std::max<int64_t>((int64_t)(win_lo / std::max<size_t>(per_band, 1)), min_grp), 1);
  int64_t g_hi = std::max<int64_t>((int64_t)(win_hi / std::max<size_t>(per_band, 1)), g_lo);
  g_hi = std::min<int64_t>(g_hi, 4096);
  g_lo = std::min<int64_t>(g_lo, g_hi);
  int64_t grp = g_hi;
  double best_eff = -1.0;
  for (int64_t c = g_lo; c <= g_hi; ++c) {
    const int64_t ctas = c * n3, waves = (ctas + slots - 1) / slots;
    const double eff = (double)ctas / (double)(waves * slots);
    if (eff >= best_eff + 0.005 || (eff >= best_eff - 0.005 && c > grp && eff >= 0.97)) { best_eff = std::max(eff, best_eff); grp = c; }
  }
  h->band_group = (int)grp;
  if (const char* e = getenv("PWH_BAND_GROUP")) {   // measurement aid (include/pwham.h): fixed group size
    const long v = strtol(e, nullptr, 10);
    if (v >= 1 && v <= 4096) h->band_group = (int)v;
  }
  h->lways = env_on("PWH_LOCAL_ONE_STREAM") ? 1 : 2;
  h->lbufs = h->lways;
  h->ltune = h->lways == 2 && !env_on("PWH_LOCAL_TWO_STREAMS");
  if (h->ltune)
    for (auto& pr : h->ltune_ev)
      for (cudaEvent_t& e : pr) CUDA_TRY(cudaEventCreate(&e));
  if (h->lways == 2) {
    for (int i = 0; i < 2; ++i) {
      CUDA_TRY(cudaStreamCreateWithFlags(&h->ls[i], cudaStreamNonBlocking));
      CUDA_TRY(cudaEventCreateWithFlags(&h->lev_join[i], cudaEventDisableTiming));
    }
    CUDA_TRY(cudaEventCreateWithFlags(&h->lev_fork, cudaEventDisableTiming));
  }

  CUDA_TRY(cudaStreamSynchronize(st));
  return PWH_OK;
}

extern "C" int pwh_ham_setup(pwh_ham** out, const double lattice[9], const double kpt[3], const int32_t fft_dims[3],
                             int64_t npw, const int32_t* gvec, const double* vloc, int64_t nproj, const pwh_c128* proj,
                             int64_t ldp, const double* dij, void* stream) {
  if (!out) return fail(PWH_EINVAL, "out is null");
  *out = nullptr;
  if (!lattice || !kpt || !fft_dims || !gvec || !vloc) return fail(PWH_EINVAL, "null argument");
  if (npw < 1 || npw > (int64_t)INT32_MAX / 2) return fail(PWH_EINVAL, "npw = %lld out of range", (long long)npw);
  if (nproj < 0 || nproj > (int64_t)INT32_MAX / 2) return fail(PWH_EINVAL, "nproj out of range");
  if (nproj > 0 && (!proj || !dij)) return fail(PWH_EINVAL, "proj / dij null with nproj > 0");
  if (nproj > 0 && ldp < npw) return fail(PWH_EINVAL, "ldp < npw");
  if ((int64_t)fft_dims[0] * fft_dims[1] * fft_dims[2] < npw) return fail(PWH_EINVAL, "more plane waves than box points");
  pwh_ham* h = new (std::nothrow) pwh_ham();
  if (!h) return fail(PWH_ENOMEM, "out of host memory");
  const int rc = setup_impl(h, lattice, kpt, fft_dims, npw, gvec, vloc, nproj, proj, ldp, dij, (cudaStream_t)stream);
  if (rc != PWH_OK) {
    pwh_ham_destroy(h);
    return rc;
  }
  *out = h;
  return PWH_OK;
}

namespace pwh {
const double* ham_kin(const pwh_ham* h) { return h->lp.kin; }
}  // namespace pwh

extern "C" int pwh_ham_info(const pwh_ham* h, int64_t info[8]) {
  if (!h || !info) return fail(PWH_EINVAL, "null argument");
  info[0] = h->npw; info[1] = h->nproj; info[2] = h->n1; info[3] = h->n2; info[4] = h->n3;
  info[5] = h->lp.ncols; info[6] = h->lp.nxl; info[7] = h->band_group;
  return PWH_OK;
}

extern "C" int pwh_ham_kernels(const pwh_ham* h, char* buf, size_t n) {
  if (!h || !buf || n == 0) return fail(PWH_EINVAL, "null argument");
  std::string s;
  if (h->fast) {
    s += h->zw ? "kz_scatter_zinv " : "kf_scatter_zinv ";
    s += h->v2 ? "kv2_plane " : "kf_plane ";
    s += h->zw ? "kz_zfwd_gather " : "kf_zfwd_gather ";
  } else {
    s += "k_scatter_zinv k_plane k_zfwd_gather ";
  }
  if (h->nproj > 0) s += h->pmaps.ok ? "zgemm3m_tma" : "zgemm3m";
  if (h->paw) s += " paw_blocks";
  s += h->ltune ? " local_streams:undecided" : (h->lways == 2 ? " local_streams:2" : " local_streams:1");
  snprintf(buf, n, "%s", s.c_str());
  return PWH_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// workspace
// ---------------------------------------------------------------------------------------------------------------
struct WsLayout {
  size_t colbuf, colbuf_bytes, cmat, part, y1, y2, total;
  int64_t ldw;
  int group;
};

// Every term is non-decreasing in nband (the split-K scratch is sized for the worst narrower block, because the split
// count is not monotone in the number of tiles), so a workspace of pwh_workspace_bytes(ham, nband_max) serves every call
// with nband <= nband_max, as include/pwham.h promises.
static WsLayout ws_layout(const pwh_ham* h, int64_t nband) {
  WsLayout w;
  w.group = (int)std::min<int64_t>(h->band_group, std::max<int64_t>(nband, 1));
  w.ldw = (int64_t)align_up((size_t)h->npw, 16);
  size_t off = 0;
  w.colbuf_bytes = align_up((size_t)w.group * h->n3 * h->lp.ncols_pad * sizeof(c128), 256);
  w.colbuf = off; off += (size_t)h->lbufs * w.colbuf_bytes;
  // projections C = P^H Y; with PAW blocks also blockdiag(D) C and blockdiag(Q) C (or K C)
  w.cmat = off;   off += (h->paw ? 3 : 1) * align_up((size_t)std::max<int64_t>(h->nproj, 1) * nband * sizeof(c128), 256);
  w.part = off;   off += align_up(h->nproj > 0 ? zgemm_cn_workspace_upto(h->nproj, nband, h->npw) : 16, 256);
  w.y1 = off;     off += align_up((size_t)w.ldw * nband * sizeof(c128), 256);
  w.y2 = off;     off += align_up((size_t)w.ldw * nband * sizeof(c128), 256);
  w.total = off;
  return w;
}

extern "C" size_t pwh_workspace_bytes(const pwh_ham* h, int64_t nband_max) {
  if (!h || nband_max < 0) return 0;
  return ws_layout(h, std::max<int64_t>(nband_max, 1)).total;
}

// out = alpha * ((H - c) y) - beta * yprev   for nband bands.  `out` may be the buffer of `yprev` (three-term recurrence
// in place over Y_{j-1}) or, when yprev is null, the buffer of `y` itself: every kernel that writes out[g] has read y[g]
// and yprev[g] in the same thread before, and the projector coefficients P^H y are complete before the first write.
static int h_step(pwh_ham* h, int64_t nband, const c128* y, int64_t ldy, const c128* yprev, int64_t ldprev, c128* out,
                  int64_t ldout, double alpha, double cshift, double beta, unsigned char* ws, const WsLayout& w,
                  cudaStream_t st) {
  c128* colbuf = reinterpret_cast<c128*>(ws + w.colbuf);
  c128* cmat = reinterpret_cast<c128*>(ws + w.cmat);
  const size_t cmat_sz = align_up((size_t)std::max<int64_t>(h->nproj, 1) * nband * sizeof(c128), 256);
  c128* cd = cmat;                                          // D C: what the second ZGEMM multiplies P with
  if (h->nproj > 0) {
    NvtxRange r("pwh:nonlocal:C=D.P^H.Y");
    launch_zgemm_cn(h->nproj, nband, h->npw, h->proj, h->ldp, y, ldy, h->paw ? nullptr : h->dij, cmat, h->nproj,
                    ws + w.part, st, &h->pmaps);
    if (h->paw) {   // per-atom dense blocks D^R
      cd = reinterpret_cast<c128*>(ws + w.cmat + cmat_sz);
      launch_blockdiag_apply(h->nproj, nband, h->blk_of, h->blk_lo, h->boff, h->dblk, cmat, h->nproj, cd, h->nproj, st);
    }
  }
  {
    NvtxRange r("pwh:local+kinetic+recurrence");
    // two-way interleave of the band groups (bands never interact); one stream while the per-launch
    // profile is on, so that the per-kernel event times are those of kernels running alone
    int ways = (h->lways == 2 && nband > w.group && !g_prof_on.load(std::memory_order_relaxed)) ? 2 : 1;
    int tune_slot = -1;
    if (ways == 2 && h->ltune) {
      if (h->ltune_calls < 4 && (h->ltune_calls == 0 || nband == h->ltune_nband)) {
        h->ltune_nband = nband;
        tune_slot = h->ltune_calls++;
        ways = (tune_slot & 1) ? 1 : 2;
        CUDA_TRY(cudaEventRecord(h->ltune_ev[tune_slot][0], st));
      } else if (h->ltune_calls >= 4) {
        bool done = true;
        for (int i = 0; i < 4 && done; ++i) done = cudaEventQuery(h->ltune_ev[i][1]) == cudaSuccess;
        if (done) {
          float t[4] = {0, 0, 0, 0};
          for (int i = 0; i < 4; ++i) CUDA_TRY(cudaEventElapsedTime(&t[i], h->ltune_ev[i][0], h->ltune_ev[i][1]));
          // slots 0, 2: two streams; 1, 3: one stream.  The first slot also pays first-touch costs: compare the second pair.
          h->lways = t[3] < t[2] ? 1 : 2;
          h->ltune = false;
          ways = h->lways;
        } else {
          (void)cudaGetLastError();   // cudaErrorNotReady is not an error
        }
      } else {
        h->ltune_calls = 0;            // a different block size: start over with this one
      }
    }
    if (ways == 2) {
      CUDA_TRY(cudaEventRecord(h->lev_fork, st));
      for (int i = 0; i < 2; ++i) CUDA_TRY(cudaStreamWaitEvent(h->ls[i], h->lev_fork, 0));
    }
    // groups of equal size (they differ by at most one band): no short last group
    const int64_t ngroups = (nband + w.group - 1) / w.group, gbase = nband / ngroups, grem = nband % ngroups;
    int64_t b0 = 0;
    for (int64_t gi = 0; gi < ngroups; ++gi) {
      const int nb = (int)(gbase + (gi < grem ? 1 : 0));
      cudaStream_t ls = ways == 2 ? h->ls[gi & 1] : st;
      c128* cb = ways == 2 ? reinterpret_cast<c128*>(ws + w.colbuf + (size_t)(gi & 1) * w.colbuf_bytes) : colbuf;
      if (h->fast) {
        if (h->zw) launch_zw_scatter_zinv(h->zp, y + b0 * ldy, ldy, cb, nb, ls);
        else launch_fast_scatter_zinv(h->fp, y + b0 * ldy, ldy, cb, nb, ls);
        if (h->v2) launch_v2_plane(h->vp, cb, nb, ls);
        else launch_fast_plane(h->fp, cb, nb, ls);
        if (h->zw)
          launch_zw_zfwd_gather(h->zp, cb, y + b0 * ldy, ldy, yprev ? yprev + b0 * ldprev : nullptr, ldprev,
                                out + b0 * ldout, ldout, alpha, cshift, yprev ? beta : 0.0, nb, ls);
        else
          launch_fast_zfwd_gather(h->fp, cb, y + b0 * ldy, ldy, yprev ? yprev + b0 * ldprev : nullptr, ldprev,
                                  out + b0 * ldout, ldout, alpha, cshift, yprev ? beta : 0.0, nb, ls);
      } else {
        launch_scatter_zinv(h->lp, y + b0 * ldy, ldy, cb, nb, ls);
        launch_plane(h->lp, cb, nb, ls);
        launch_zfwd_gather(h->lp, cb, y + b0 * ldy, ldy, yprev ? yprev + b0 * ldprev : nullptr, ldprev,
                           out + b0 * ldout, ldout, alpha, cshift, yprev ? beta : 0.0, nb, ls);
      }
      b0 += nb;
    }
    if (ways == 2)
      for (int i = 0; i < 2; ++i) {
        CUDA_TRY(cudaEventRecord(h->lev_join[i], h->ls[i]));
        CUDA_TRY(cudaStreamWaitEvent(st, h->lev_join[i], 0));
      }
    if (tune_slot >= 0) CUDA_TRY(cudaEventRecord(h->ltune_ev[tune_slot][1], st));
  }
  if (h->nproj > 0) {
    NvtxRange r("pwh:nonlocal:Y+=a.P.C");
    launch_zgemm_nn(h->npw, nband, h->nproj, alpha, h->proj, h->ldp, cd, h->nproj, out, ldout, true, st, &h->pmaps);
  }
  CUDA_TRY(cudaGetLastError());
  return PWH_OK;
}

static int check_ws(const pwh_ham* h, int64_t nband, void* ws, size_t ws_bytes) {
  if (!ws) return fail(PWH_EINVAL, "workspace is null");
  if ((uintptr_t)ws % 256 != 0) return fail(PWH_EINVAL, "workspace must be 256-byte aligned");
  const size_t need = ws_layout(h, nband).total;
  if (ws_bytes < need) return fail(PWH_EINVAL, "workspace too small: %zu < %zu bytes", ws_bytes, need);
  return PWH_OK;
}

// do the address ranges of two column-major blocks (npw x nband, leading dimensions lda / ldb) intersect?
static bool blocks_overlap(const void* a, int64_t lda, const void* b, int64_t ldb, int64_t npw, int64_t nband) {
  const uintptr_t a0 = (uintptr_t)a, a1 = a0 + ((size_t)(nband - 1) * lda + npw) * sizeof(c128);
  const uintptr_t b0 = (uintptr_t)b, b1 = b0 + ((size_t)(nband - 1) * ldb + npw) * sizeof(c128);
  return a0 < b1 && b0 < a1;
}

extern "C" int pwh_apply_h(pwh_ham* h, int64_t nband, const pwh_c128* psi, int64_t ldpsi, pwh_c128* hpsi, int64_t ldh,
                           void* ws, size_t ws_bytes, void* stream) {
  if (!h) return fail(PWH_EINVAL, "handle is null");
  if (nband < 0) return fail(PWH_EINVAL, "nband < 0");
  if (nband == 0) return PWH_OK;
  if (!psi || !hpsi) return fail(PWH_EINVAL, "psi / hpsi null");
  if (ldpsi < h->npw || ldh < h->npw) return fail(PWH_EINVAL, "leading dimension smaller than npw");
  int rc = check_ws(h, nband, ws, ws_bytes);
  if (rc) return rc;
  if (blocks_overlap(psi, ldpsi, hpsi, ldh, h->npw, nband)) return fail(PWH_EINVAL, "psi and hpsi overlap");
  NvtxRange r("pwh_apply_h");
  const WsLayout w = ws_layout(h, nband);
  return h_step(h, nband, reinterpret_cast<const c128*>(psi), ldpsi, nullptr, 0, reinterpret_cast<c128*>(hpsi), ldh, 1.0,
                0.0, 0.0, reinterpret_cast<unsigned char*>(ws), w, (cudaStream_t)stream);
}

extern "C" int pwh_cheb_filter(pwh_ham* h, int64_t nband, pwh_c128* psi, int64_t ld, int degree, double a, double b,
                               double a0, void* ws, size_t ws_bytes, void* stream) {
  if (!h) return fail(PWH_EINVAL, "handle is null");
  if (nband < 0) return fail(PWH_EINVAL, "nband < 0");
  if (degree < 0) return fail(PWH_EINVAL, "degree < 0");
  if (!(b > a)) return fail(PWH_EINVAL, "need b > a");
  if (!(a0 < a)) return fail(PWH_EINVAL, "need a0 < a");
  if (nband == 0 || degree == 0) return PWH_OK;
  if (!psi) return fail(PWH_EINVAL, "psi null");
  if (ld < h->npw) return fail(PWH_EINVAL, "ld < npw");
  int rc = check_ws(h, nband, ws, ws_bytes);
  if (rc) return rc;
  NvtxRange r("pwh_cheb_filter");
  const WsLayout w = ws_layout(h, nband);
  unsigned char* wsb = reinterpret_cast<unsigned char*>(ws);
  cudaStream_t st = (cudaStream_t)stream;
  c128* buf[3] = {reinterpret_cast<c128*>(psi), reinterpret_cast<c128*>(wsb + w.y1), reinterpret_cast<c128*>(wsb + w.y2)};
  const int64_t lds[3] = {ld, w.ldw, w.ldw};
  const double e = 0.5 * (b - a), c = 0.5 * (b + a), sigma1 = e / (a0 - c);
  // Where Y_j lives (0 = psi, 1 and 2 = workspace), chosen so that Y_degree lands in psi without a final copy:
  // from the second (even degree) or fourth (odd degree) step on, Y_{j+1} is written over Y_{j-1}, which the
  // recurrence reads for the last time in that very step; Y_1 of a degree-1 filter is written over Y_0 itself.
  std::vector<int> where((size_t)degree + 1, 0);
  if (degree % 2 == 0) {
    where[1] = 1;
    for (int j = 2; j <= degree; ++j) where[j] = where[j - 2];
  } else if (degree >= 3) {
    where[1] = 1; where[2] = 2; where[3] = 0;
    for (int j = 4; j <= degree; ++j) where[j] = where[j - 2];
  }
  double sigma = sigma1;
  // Y_1 = (sigma_1/e) (H - c) Y_0
  rc = h_step(h, nband, buf[0], lds[0], nullptr, 0, buf[where[1]], lds[where[1]], sigma1 / e, c, 0.0, wsb, w, st);
  if (rc) return rc;
  for (int j = 1; j < degree; ++j) {
    const double sigma_new = 1.0 / (2.0 / sigma1 - sigma);
    const int ip = where[j - 1], ic = where[j], io = where[j + 1];
    rc = h_step(h, nband, buf[ic], lds[ic], buf[ip], lds[ip], buf[io], lds[io], 2.0 * sigma_new / e, c,
                sigma * sigma_new, wsb, w, st);
    if (rc) return rc;
    sigma = sigma_new;
  }
  return PWH_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// electronic density (Algorithm 3 step 10)
// ---------------------------------------------------------------------------------------------------------------
struct DensLayout { size_t colbuf, acc, total; int group; };
static DensLayout dens_layout(const pwh_ham* h, int64_t nband) {
  DensLayout d;
  d.group = (int)std::min<int64_t>(h->band_group, std::max<int64_t>(nband, 1));
  size_t off = 0;
  d.colbuf = off; off += align_up((size_t)d.group * h->n3 * h->lp.ncols_pad * sizeof(c128), 256);
  d.acc = off;    off += align_up((size_t)h->n1 * h->n2 * h->n3 * sizeof(double), 256);
  d.total = off;
  return d;
}

extern "C" size_t pwh_density_workspace_bytes(const pwh_ham* h, int64_t nband_max) {
  if (!h || nband_max < 0) return 0;
  return dens_layout(h, std::max<int64_t>(nband_max, 1)).total;
}

extern "C" int pwh_density_accumulate(pwh_ham* h, int64_t nband, const pwh_c128* psi, int64_t ld, const double* occ,
                                      double weight, double* rho, void* ws, size_t ws_bytes, void* stream) {
  if (!h) return fail(PWH_EINVAL, "handle is null");
  if (nband < 0) return fail(PWH_EINVAL, "nband < 0");
  if (nband == 0) return PWH_OK;
  if (!psi || !occ || !rho) return fail(PWH_EINVAL, "psi / occ / rho null");
  if (ld < h->npw) return fail(PWH_EINVAL, "ld < npw");
  if (!ws || (uintptr_t)ws % 256 != 0) return fail(PWH_EINVAL, "workspace null or not 256-byte aligned");
  const DensLayout d = dens_layout(h, nband);
  if (ws_bytes < d.total) return fail(PWH_EINVAL, "workspace too small: %zu < %zu bytes", ws_bytes, d.total);
  NvtxRange r("pwh_density_accumulate");
  cudaStream_t st = (cudaStream_t)stream;
  unsigned char* wsb = reinterpret_cast<unsigned char*>(ws);
  c128* colbuf = reinterpret_cast<c128*>(wsb + d.colbuf);
  double* acc = reinterpret_cast<double*>(wsb + d.acc);
  const c128* y = reinterpret_cast<const c128*>(psi);
  CUDA_TRY(cudaMemsetAsync(acc, 0, (size_t)h->n1 * h->n2 * h->n3 * sizeof(double), st));
  for (int64_t b0 = 0; b0 < nband; b0 += d.group) {
    const int nb = (int)std::min<int64_t>(d.group, nband - b0);
    if (h->fast) {
      if (h->zw) launch_zw_scatter_zinv(h->zp, y + b0 * ld, ld, colbuf, nb, st);
      else launch_fast_scatter_zinv(h->fp, y + b0 * ld, ld, colbuf, nb, st);
      launch_fast_density_plane(h->fp, colbuf, nb, occ + b0, acc, st);
    } else {
      launch_scatter_zinv(h->lp, y + b0 * ld, ld, colbuf, nb, st);
      launch_density_plane(h->lp, colbuf, nb, occ + b0, acc, st);
    }
  }
  if (h->fast) launch_fast_density_unslot(h->fp, acc, weight, rho, st);
  else launch_density_unpermute(h->lp, acc, h->dnat[0], h->dnat[1], h->dnat[2], weight, rho, st);
  CUDA_TRY(cudaGetLastError());
  return PWH_OK;
}

extern "C" size_t pwh_gram_workspace_bytes(int64_t npw, int64_t nx, int64_t ny) {
  if (npw < 1 || nx < 1 || ny < 1) return 256;
  // the Hermitian variant computes fewer tiles and may choose more K splits: size for both
  size_t need = zgemm_cn_workspace(nx, ny, npw, false);
  if (nx == ny) need = std::max(need, zgemm_cn_workspace(nx, ny, npw, true));
  return align_up(need, 256);
}

static int gram_impl(int64_t npw, int64_t nx, const pwh_c128* X, int64_t ldx, int64_t ny, const pwh_c128* Y, int64_t ldy,
                     pwh_c128* G, int64_t ldg, void* ws, size_t ws_bytes, void* stream, bool herm) {
  if (npw < 1 || nx < 0 || ny < 0) return fail(PWH_EINVAL, "bad sizes");
  if (herm && nx != ny) return fail(PWH_EINVAL, "a Hermitian Gram matrix needs nx == ny");
  if (nx == 0 || ny == 0) return PWH_OK;
  if (nx > INT32_MAX / 2 || ny > INT32_MAX / 2) return fail(PWH_EINVAL, "nx / ny too large");
  if (!X || !Y || !G) return fail(PWH_EINVAL, "null argument");
  if (ldx < npw || ldy < npw || ldg < nx) return fail(PWH_EINVAL, "leading dimension too small");
  if (!ws || (uintptr_t)ws % 256 != 0) return fail(PWH_EINVAL, "workspace null or not 256-byte aligned");
  if (ws_bytes < pwh_gram_workspace_bytes(npw, nx, ny)) return fail(PWH_EINVAL, "workspace too small");
  CUDA_TRY(zgemm_init());
  NvtxRange r(herm ? "pwh_gram_herm" : "pwh_gram");
  launch_zgemm_cn(nx, ny, npw, reinterpret_cast<const c128*>(X), ldx, reinterpret_cast<const c128*>(Y), ldy, nullptr,
                  reinterpret_cast<c128*>(G), ldg, ws, (cudaStream_t)stream, nullptr, herm);
  CUDA_TRY(cudaGetLastError());
  return PWH_OK;
}

extern "C" int pwh_gram(int64_t npw, int64_t nx, const pwh_c128* X, int64_t ldx, int64_t ny, const pwh_c128* Y,
                        int64_t ldy, pwh_c128* G, int64_t ldg, void* ws, size_t ws_bytes, void* stream) {
  return gram_impl(npw, nx, X, ldx, ny, Y, ldy, G, ldg, ws, ws_bytes, stream, false);
}

extern "C" int pwh_gram_herm(int64_t npw, int64_t n, const pwh_c128* X, int64_t ldx, const pwh_c128* Y, int64_t ldy,
                             pwh_c128* G, int64_t ldg, void* ws, size_t ws_bytes, void* stream) {
  return gram_impl(npw, n, X, ldx, n, Y, ldy, G, ldg, ws, ws_bytes, stream, true);
}

// ---------------------------------------------------------------------------------------------------------------
// PAW-style generalised problem H Psi = Lambda S Psi
// ---------------------------------------------------------------------------------------------------------------
extern "C" int pwh_ham_set_paw(pwh_ham* h, int64_t nblocks, const int32_t* offsets, const pwh_c128* dblocks,
                               const pwh_c128* qblocks, int32_t* info, void* stream) {
  if (!h) return fail(PWH_EINVAL, "handle is null");
  if (h->nproj < 1) return fail(PWH_EINVAL, "the handle has no projectors");
  if (nblocks < 1 || !offsets || !dblocks || !qblocks || !info) return fail(PWH_EINVAL, "null argument or nblocks < 1");
  if (offsets[0] != 0 || offsets[nblocks] != h->nproj) return fail(PWH_EINVAL, "offsets must run from 0 to nproj");
  for (int64_t r = 0; r < nblocks; ++r)
    if (offsets[r + 1] <= offsets[r]) return fail(PWH_EINVAL, "offsets must increase");
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t J = h->nproj;
  std::vector<int> blk_of((size_t)J), blk_lo((size_t)nblocks + 1);
  std::vector<int64_t> boff((size_t)nblocks);
  int64_t tot = 0;
  for (int64_t r = 0; r < nblocks; ++r) {
    blk_lo[r] = offsets[r];
    boff[r] = tot;
    const int64_t n = offsets[r + 1] - offsets[r];
    tot += n * n;
    for (int64_t i = offsets[r]; i < offsets[r + 1]; ++i) blk_of[i] = (int)r;
  }
  blk_lo[nblocks] = (int)J;
  int rc;
  const int* d_of; const int* d_lo; const int64_t* d_off;
  if ((rc = upload(h, blk_of, &d_of, st)) || (rc = upload(h, blk_lo, &d_lo, st)) || (rc = upload(h, boff, &d_off, st))) return rc;
  c128 *db = nullptr, *qb = nullptr, *km = nullptr;
  CUDA_TRY(cudaMalloc(&db, tot * sizeof(c128))); h->allocs.push_back(db);
  CUDA_TRY(cudaMalloc(&qb, tot * sizeof(c128))); h->allocs.push_back(qb);
  CUDA_TRY(cudaMalloc(&km, (size_t)J * J * sizeof(c128))); h->allocs.push_back(km);
  CUDA_TRY(cudaMemcpyAsync(db, dblocks, tot * sizeof(c128), cudaMemcpyDeviceToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(qb, qblocks, tot * sizeof(c128), cudaMemcpyDeviceToDevice, st));
  // K of S^-1 = I - P K P^H (Woodbury), through two Cholesky factorisations so that only Hermitian
  // positive definite matrices are factored:  G = P^H P = U^H U,  A = U Q U^H,  I + A = V^H V,  W = U^-1,  Z = V^-1,
  //   K = W (I - Z Z^H) W^H = W W^H - (W Z)(W Z)^H        [ = G^-1 - (G + G Q G)^-1 ]
  const size_t mat = align_up((size_t)J * J * sizeof(c128), 256);
  const size_t part = align_up(std::max(zgemm_cn_workspace(J, J, h->npw, true), zgemm_cn_workspace(J, J, J, true)), 256);
  unsigned char* scr = nullptr;
  CUDA_TRY(cudaMalloc(&scr, 5 * mat + part + 256));
  c128* G = (c128*)scr; c128* W = (c128*)(scr + mat); c128* T1 = (c128*)(scr + 2 * mat); c128* T2 = (c128*)(scr + 3 * mat);
  c128* T3 = (c128*)(scr + 4 * mat);
  void* pws = scr + 5 * mat;
  int* pinfo = (int*)(scr + 5 * mat + part);
  const int n = (int)J;
  cudaError_t ce = rr_kernels_init();
  if (ce == cudaSuccess) ce = zgemm_init();
  if (ce == cudaSuccess) {
    CUDA_TRY(cudaMemsetAsync(info, 0, sizeof(int), st));
    launch_zgemm_cn(J, J, h->npw, h->proj, h->ldp, h->proj, h->ldp, nullptr, G, J, pws, st, &h->pmaps, true);   // G = P^H P
    launch_hermitise(n, G, J, st);
    launch_potrf_upper(n, G, J, pinfo, st);                                  // G <- U
    launch_merge_info(pinfo, info, st);
    launch_trinv_upper(n, G, J, W, J, st);                                   // W = U^-1
    launch_blocks_to_dense(J, d_of, d_lo, d_off, qb, T1, J, st);             // T1 = Q
    launch_conj_transpose(n, G, J, T2, J, st);                               // T2 = U^H
    launch_zgemm_nn(J, J, J, 1.0, T1, J, T2, J, T3, J, false, st);           // T3 = Q U^H
    launch_zgemm_nn(J, J, J, 1.0, G, J, T3, J, T1, J, false, st);            // T1 = A = U Q U^H
    launch_mat_axpby(n, 1.0, T1, J, 0.0, nullptr, 0, 1.0, st);               // T1 = I + A
    launch_hermitise(n, T1, J, st);
    launch_potrf_upper(n, T1, J, pinfo, st);                                 // T1 <- V
    launch_merge_info(pinfo, info, st);
    launch_trinv_upper(n, T1, J, T2, J, st);                                 // T2 = Z = V^-1
    launch_zgemm_nn(J, J, J, 1.0, W, J, T2, J, T3, J, false, st);            // T3 = W Z
    launch_conj_transpose(n, T3, J, T1, J, st);                              // T1 = (W Z)^H
    launch_conj_transpose(n, W, J, T2, J, st);                               // T2 = W^H
    launch_zgemm_cn(J, J, J, T2, J, T2, J, nullptr, km, J, pws, st, nullptr, true);   // K = W W^H
    launch_zgemm_cn(J, J, J, T1, J, T1, J, nullptr, T3, J, pws, st, nullptr, true);   // T3 = (W Z)(W Z)^H
    launch_mat_axpby(n, 1.0, km, J, -1.0, T3, J, 0.0, st);
    launch_hermitise(n, km, J, st);
    ce = cudaGetLastError();
  }
  const cudaError_t cs = cudaStreamSynchronize(st);
  cudaFree(scr);
  CUDA_TRY(ce);
  CUDA_TRY(cs);
  h->blk_of = const_cast<int*>(d_of); h->blk_lo = const_cast<int*>(d_lo); h->boff = const_cast<int64_t*>(d_off);
  h->dblk = db; h->qblk = qb; h->kmat = km;
  h->paw = true;
  return PWH_OK;
}

// H psi and S psi from one set of projections (HX_SX); either output may be null
extern "C" int pwh_apply_hs(pwh_ham* h, int64_t nband, const pwh_c128* psi, int64_t ldpsi, pwh_c128* hpsi, int64_t ldh,
                            pwh_c128* spsi, int64_t lds, void* ws, size_t ws_bytes, void* stream) {
  if (!h) return fail(PWH_EINVAL, "handle is null");
  if (!h->paw) return fail(PWH_EINVAL, "pwh_ham_set_paw has not been called on this handle");
  if (nband < 0) return fail(PWH_EINVAL, "nband < 0");
  if (nband == 0) return PWH_OK;
  if (!psi || (!hpsi && !spsi)) return fail(PWH_EINVAL, "psi null or no output");
  if (ldpsi < h->npw || (hpsi && ldh < h->npw) || (spsi && lds < h->npw)) return fail(PWH_EINVAL, "leading dimension smaller than npw");
  int rc = check_ws(h, nband, ws, ws_bytes);
  if (rc) return rc;
  if (hpsi && blocks_overlap(psi, ldpsi, hpsi, ldh, h->npw, nband)) return fail(PWH_EINVAL, "psi and hpsi overlap");
  if (spsi && blocks_overlap(psi, ldpsi, spsi, lds, h->npw, nband)) return fail(PWH_EINVAL, "psi and spsi overlap");
  NvtxRange r("pwh_apply_hs");
  cudaStream_t st = (cudaStream_t)stream;
  const WsLayout w = ws_layout(h, nband);
  unsigned char* wsb = reinterpret_cast<unsigned char*>(ws);
  if (hpsi) {   // computes C = P^H psi into cmat on the way
    rc = h_step(h, nband, (const c128*)psi, ldpsi, nullptr, 0, (c128*)hpsi, ldh, 1.0, 0.0, 0.0, wsb, w, st);
    if (rc) return rc;
  }
  if (spsi) {
    c128* cmat = reinterpret_cast<c128*>(wsb + w.cmat);
    const size_t cmat_sz = align_up((size_t)h->nproj * nband * sizeof(c128), 256);
    c128* cq = reinterpret_cast<c128*>(wsb + w.cmat + 2 * cmat_sz);
    if (!hpsi)
      launch_zgemm_cn(h->nproj, nband, h->npw, h->proj, h->ldp, (const c128*)psi, ldpsi, nullptr, cmat, h->nproj, wsb + w.part,
                      st, &h->pmaps);
    launch_blockdiag_apply(h->nproj, nband, h->blk_of, h->blk_lo, h->boff, h->qblk, cmat, h->nproj, cq, h->nproj, st);
    CUDA_TRY(cudaMemcpy2DAsync(spsi, (size_t)lds * sizeof(c128), psi, (size_t)ldpsi * sizeof(c128), (size_t)h->npw * sizeof(c128),
                               (size_t)nband, cudaMemcpyDeviceToDevice, st));
    launch_zgemm_nn(h->npw, nband, h->nproj, 1.0, h->proj, h->ldp, cq, h->nproj, (c128*)spsi, lds, true, st, &h->pmaps);
    CUDA_TRY(cudaGetLastError());
  }
  return PWH_OK;
}

// x <- S^-1 x = x - P K (P^H x) in place
static int sinv_inplace(pwh_ham* h, int64_t nband, c128* x, int64_t ldx, unsigned char* wsb, const WsLayout& w, cudaStream_t st) {
  c128* cmat = reinterpret_cast<c128*>(wsb + w.cmat);
  const size_t cmat_sz = align_up((size_t)h->nproj * nband * sizeof(c128), 256);
  c128* ck = reinterpret_cast<c128*>(wsb + w.cmat + 2 * cmat_sz);
  launch_zgemm_cn(h->nproj, nband, h->npw, h->proj, h->ldp, x, ldx, nullptr, cmat, h->nproj, wsb + w.part, st, &h->pmaps);
  launch_zgemm_nn(h->nproj, nband, h->nproj, 1.0, h->kmat, h->nproj, cmat, h->nproj, ck, h->nproj, false, st);
  launch_zgemm_nn(h->npw, nband, h->nproj, -1.0, h->proj, h->ldp, ck, h->nproj, x, ldx, true, st, &h->pmaps);
  CUDA_TRY(cudaGetLastError());
  return PWH_OK;
}

extern "C" int pwh_apply_sinv(pwh_ham* h, int64_t nband, pwh_c128* x, int64_t ldx, void* ws, size_t ws_bytes, void* stream) {
  if (!h) return fail(PWH_EINVAL, "handle is null");
  if (!h->paw) return fail(PWH_EINVAL, "pwh_ham_set_paw has not been called on this handle");
  if (nband < 0) return fail(PWH_EINVAL, "nband < 0");
  if (nband == 0) return PWH_OK;
  if (!x || ldx < h->npw) return fail(PWH_EINVAL, "x null or ldx < npw");
  int rc = check_ws(h, nband, ws, ws_bytes);
  if (rc) return rc;
  NvtxRange r("pwh_apply_sinv");
  return sinv_inplace(h, nband, (c128*)x, ldx, reinterpret_cast<unsigned char*>(ws), ws_layout(h, nband), (cudaStream_t)stream);
}

// the scaled Chebyshev filter of S^-1 H (Algorithm 12 lines 4-8): per degree T = H Y_j, T <- S^-1 T, axpy
extern "C" int pwh_cheb_filter_gen(pwh_ham* h, int64_t nband, pwh_c128* psi, int64_t ld, int degree, double a, double b,
                                   double a0, void* ws, size_t ws_bytes, void* stream) {
  if (!h) return fail(PWH_EINVAL, "handle is null");
  if (!h->paw) return fail(PWH_EINVAL, "pwh_ham_set_paw has not been called on this handle");
  if (nband < 0) return fail(PWH_EINVAL, "nband < 0");
  if (degree < 0) return fail(PWH_EINVAL, "degree < 0");
  if (!(b > a)) return fail(PWH_EINVAL, "need b > a");
  if (!(a0 < a)) return fail(PWH_EINVAL, "need a0 < a");
  if (nband == 0 || degree == 0) return PWH_OK;
  if (!psi) return fail(PWH_EINVAL, "psi null");
  if (ld < h->npw) return fail(PWH_EINVAL, "ld < npw");
  int rc = check_ws(h, nband, ws, ws_bytes);
  if (rc) return rc;
  NvtxRange r("pwh_cheb_filter_gen");
  const WsLayout w = ws_layout(h, nband);
  unsigned char* wsb = reinterpret_cast<unsigned char*>(ws);
  cudaStream_t st = (cudaStream_t)stream;
  c128* buf[3] = {reinterpret_cast<c128*>(psi), reinterpret_cast<c128*>(wsb + w.y1), reinterpret_cast<c128*>(wsb + w.y2)};
  const int64_t lds[3] = {ld, w.ldw, w.ldw};
  const double e = 0.5 * (b - a), c = 0.5 * (b + a), sigma1 = e / (a0 - c);
  // where Y_j lives; T = S^-1 H Y_j goes to the one buffer that holds neither Y_j nor Y_{j-1}, and Y_{j+1} is written either
  // over T or over Y_{j-1} (the axpy is entry by entry), chosen so that Y_degree lands in psi (as in pwh_cheb_filter)
  std::vector<int> where((size_t)degree + 1, 0);
  if (degree % 2 == 0) {
    where[1] = 1;
    for (int j = 2; j <= degree; ++j) where[j] = where[j - 2];
  } else if (degree >= 3) {
    where[1] = 1; where[2] = 2; where[3] = 0;
    for (int j = 4; j <= degree; ++j) where[j] = where[j - 2];
  }
  double sigma = sigma1;
  for (int j = 0; j < degree; ++j) {
    const int ic = where[j], ip = j > 0 ? where[j - 1] : -1, io = where[j + 1];
    int it = 0;
    while (it == ic || it == ip) ++it;                 // the free buffer
    rc = h_step(h, nband, buf[ic], lds[ic], nullptr, 0, buf[it], lds[it], 1.0, 0.0, 0.0, wsb, w, st);   // T = H Y_j
    if (rc) return rc;
    if ((rc = sinv_inplace(h, nband, buf[it], lds[it], wsb, w, st))) return rc;                          // T <- S^-1 T
    double alpha, beta = 0.0;
    if (j == 0) alpha = sigma1 / e;
    else {
      const double sigma_new = 1.0 / (2.0 / sigma1 - sigma);
      alpha = 2.0 * sigma_new / e;
      beta = sigma * sigma_new;
      sigma = sigma_new;
    }
    launch_cheb_axpy(h->npw, nband, buf[it], lds[it], buf[ic], lds[ic], j > 0 ? buf[ip] : nullptr, j > 0 ? lds[ip] : 0,
                     buf[io], lds[io], alpha, c, beta, st);
  }
  CUDA_TRY(cudaGetLastError());
  return PWH_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// host-buffer entry points
// ---------------------------------------------------------------------------------------------------------------
static int ensure(void** p, size_t* have, size_t need) {
  if (*have >= need) return PWH_OK;
  if (*p) cudaFree(*p);
  *p = nullptr;
  *have = 0;
  CUDA_TRY(cudaMalloc(p, need));
  *have = need;
  return PWH_OK;
}

// Every exit of a host entry point -- success or error -- waits for the caller's stream and the two copy streams, so no
// copy into or out of the caller's host buffers is still in flight when the call returns (include/pwham.h).
static int host_finish(pwh_ham* h, cudaStream_t st, int rc) {
  const cudaError_t e0 = cudaStreamSynchronize(st);
  const cudaError_t e1 = h->cs_in ? cudaStreamSynchronize(h->cs_in) : cudaSuccess;
  const cudaError_t e2 = h->cs_out ? cudaStreamSynchronize(h->cs_out) : cudaSuccess;
  if (rc != PWH_OK) return rc;
  for (cudaError_t e : {e0, e1, e2})
    if (e != cudaSuccess) return fail(PWH_ECUDA, "stream synchronisation: %s", cudaGetErrorString(e));
  return PWH_OK;
}

static int apply_h_host_impl(pwh_ham* h, int64_t nband, const pwh_c128* psi_host, int64_t ldpsi, pwh_c128* hpsi_host,
                             int64_t ldh, cudaStream_t st) {
  const size_t blk = (size_t)h->npw * nband * sizeof(c128), row = (size_t)h->npw * sizeof(c128);
  int rc;
  if ((rc = ensure(&h->st_psi, &h->st_psi_bytes, blk))) return rc;
  if ((rc = ensure(&h->st_hpsi, &h->st_hpsi_bytes, blk))) return rc;
  if ((rc = ensure(&h->st_ws, &h->st_ws_bytes, pwh_workspace_bytes(h, nband)))) return rc;
  CUDA_TRY(cudaMemcpy2DAsync(h->st_psi, row, psi_host, (size_t)ldpsi * sizeof(c128), row, nband, cudaMemcpyHostToDevice, st));
  rc = pwh_apply_h(h, nband, (const pwh_c128*)h->st_psi, h->npw, (pwh_c128*)h->st_hpsi, h->npw, h->st_ws, h->st_ws_bytes, st);
  if (rc) return rc;
  CUDA_TRY(cudaMemcpy2DAsync(hpsi_host, (size_t)ldh * sizeof(c128), h->st_hpsi, row, row, nband, cudaMemcpyDeviceToHost, st));
  return PWH_OK;
}

extern "C" int pwh_apply_h_host(pwh_ham* h, int64_t nband, const pwh_c128* psi_host, int64_t ldpsi, pwh_c128* hpsi_host,
                                int64_t ldh, void* stream) {
  if (!h) return fail(PWH_EINVAL, "handle is null");
  if (nband < 0) return fail(PWH_EINVAL, "nband < 0");
  if (nband == 0) return PWH_OK;
  if (!psi_host || !hpsi_host) return fail(PWH_EINVAL, "null argument");
  if (ldpsi < h->npw || ldh < h->npw) return fail(PWH_EINVAL, "leading dimension smaller than npw");
  cudaStream_t st = (cudaStream_t)stream;
  return host_finish(h, st, apply_h_host_impl(h, nband, psi_host, ldpsi, hpsi_host, ldh, st));
}

static int filter_blocks(pwh_ham* h, int64_t nband, int64_t block, c128* psi_dev, int64_t ld, int degree, double a,
                         double b, double a0, cudaStream_t st) {
  if (block <= 0 || block > nband) block = nband;
  for (int64_t b0 = 0; b0 < nband; b0 += block) {
    const int64_t nb = std::min(block, nband - b0);
    int rc = pwh_cheb_filter(h, nb, (pwh_c128*)(psi_dev + b0 * ld), ld, degree, a, b, a0, h->st_ws, h->st_ws_bytes, st);
    if (rc) return rc;
  }
  return PWH_OK;
}

// The host entry points move Psi in chunks of bands on two copy streams so that the host->device copy of chunk i+1 and
// the device->host copy of chunk i-1 run under the filter of chunk i (bands never interact before gram, PAPER.md:117,
// 224): the column blocks of `block` bands when there are several, otherwise quarters of the block.
static int64_t pipeline_chunk(int64_t nband, int64_t block) {
  if (block <= 0 || block > nband) block = nband;
  if (block < nband || nband < 512) return block;
  return ((nband + 3) / 4 + 63) / 64 * 64;
}

static int pipeline_init(pwh_ham* h, size_t nevents) {
  if (!h->cs_in) CUDA_TRY(cudaStreamCreateWithFlags(&h->cs_in, cudaStreamNonBlocking));
  if (!h->cs_out) CUDA_TRY(cudaStreamCreateWithFlags(&h->cs_out, cudaStreamNonBlocking));
  while (h->evs.size() < nevents) {
    cudaEvent_t e;
    CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    h->evs.push_back(e);
  }
  return PWH_OK;
}

// H2D of all chunks on cs_in, filter of chunk c on `st` as soon as it has landed, D2H of the filtered chunk on cs_out
static int filter_pipelined(pwh_ham* h, int64_t nband, int64_t block, pwh_c128* psi_host, int64_t ld, int degree, double a,
                            double b, double a0, cudaStream_t st) {
  const int64_t chunk = pipeline_chunk(nband, block);
  const int64_t nchunks = (nband + chunk - 1) / chunk;
  const size_t row = (size_t)h->npw * sizeof(c128);
  int rc;
  if ((rc = pipeline_init(h, (size_t)(2 * nchunks + 1)))) return rc;
  c128* dev = (c128*)h->st_psi;
  CUDA_TRY(cudaEventRecord(h->evs[0], st));                       // earlier work on `st` may still use the staging buffer
  CUDA_TRY(cudaStreamWaitEvent(h->cs_in, h->evs[0], 0));
  for (int64_t c = 0; c < nchunks; ++c) {
    const int64_t b0 = c * chunk, nb = std::min(chunk, nband - b0);
    CUDA_TRY(cudaMemcpy2DAsync(dev + b0 * h->npw, row, (const c128*)psi_host + b0 * ld, (size_t)ld * sizeof(c128), row,
                               (size_t)nb, cudaMemcpyHostToDevice, h->cs_in));
    CUDA_TRY(cudaEventRecord(h->evs[1 + c], h->cs_in));
  }
  for (int64_t c = 0; c < nchunks; ++c) {
    const int64_t b0 = c * chunk, nb = std::min(chunk, nband - b0);
    CUDA_TRY(cudaStreamWaitEvent(st, h->evs[1 + c], 0));
    if ((rc = filter_blocks(h, nb, std::min<int64_t>(block > 0 ? block : nb, nb), dev + b0 * h->npw, h->npw, degree, a, b, a0, st)))
      return rc;
    CUDA_TRY(cudaEventRecord(h->evs[1 + nchunks + c], st));
    CUDA_TRY(cudaStreamWaitEvent(h->cs_out, h->evs[1 + nchunks + c], 0));
    CUDA_TRY(cudaMemcpy2DAsync((c128*)psi_host + b0 * ld, (size_t)ld * sizeof(c128), dev + b0 * h->npw, row, row, (size_t)nb,
                               cudaMemcpyDeviceToHost, h->cs_out));
  }
  return PWH_OK;
}

static int cheb_filter_host_impl(pwh_ham* h, int64_t nband, int64_t block, pwh_c128* psi_host, int64_t ld, int degree,
                                 double a, double b, double a0, cudaStream_t st) {
  const size_t blk = (size_t)h->npw * nband * sizeof(c128);
  int rc;
  if ((rc = ensure(&h->st_psi, &h->st_psi_bytes, blk))) return rc;
  if ((rc = ensure(&h->st_ws, &h->st_ws_bytes, pwh_workspace_bytes(h, std::min(block, pipeline_chunk(nband, block)))))) return rc;
  return filter_pipelined(h, nband, block, psi_host, ld, degree, a, b, a0, st);
}

extern "C" int pwh_cheb_filter_host(pwh_ham* h, int64_t nband, int64_t block, pwh_c128* psi_host, int64_t ld, int degree,
                                    double a, double b, double a0, void* stream) {
  if (!h) return fail(PWH_EINVAL, "handle is null");
  if (nband < 0) return fail(PWH_EINVAL, "nband < 0");
  if (degree < 0 || !(b > a) || !(a0 < a)) return fail(PWH_EINVAL, "bad filter parameters");
  if (nband == 0) return PWH_OK;
  if (!psi_host) return fail(PWH_EINVAL, "psi null");
  if (ld < h->npw) return fail(PWH_EINVAL, "ld < npw");
  cudaStream_t st = (cudaStream_t)stream;
  if (block <= 0 || block > nband) block = nband;
  return host_finish(h, st, cheb_filter_host_impl(h, nband, block, psi_host, ld, degree, a, b, a0, st));
}

static int sweep_host_impl(pwh_ham* h, int64_t nband, int64_t block, pwh_c128* psi_host, int64_t ld, int degree, double a,
                           double b, double a0, pwh_c128* hpsi_host, int64_t ldh, pwh_c128* G_host, int64_t ldg,
                           cudaStream_t st) {
  const size_t blk = (size_t)h->npw * nband * sizeof(c128), row = (size_t)h->npw * sizeof(c128);
  const size_t gbytes = (size_t)nband * nband * sizeof(c128);
  const size_t wsb = std::max(pwh_workspace_bytes(h, block), pwh_gram_workspace_bytes(h->npw, nband, nband));
  int rc;
  if ((rc = ensure(&h->st_psi, &h->st_psi_bytes, blk))) return rc;
  if ((rc = ensure(&h->st_hpsi, &h->st_hpsi_bytes, blk))) return rc;
  if ((rc = ensure(&h->st_g, &h->st_g_bytes, gbytes))) return rc;
  if ((rc = ensure(&h->st_ws, &h->st_ws_bytes, wsb))) return rc;
  if ((rc = filter_pipelined(h, nband, block, psi_host, ld, degree, a, b, a0, st))) return rc;
  for (int64_t b0 = 0; b0 < nband; b0 += block) {
    const int64_t nb = std::min(block, nband - b0);
    rc = pwh_apply_h(h, nb, (const pwh_c128*)((c128*)h->st_psi + b0 * h->npw), h->npw,
                     (pwh_c128*)((c128*)h->st_hpsi + b0 * h->npw), h->npw, h->st_ws, h->st_ws_bytes, st);
    if (rc) return rc;
  }
  // Psi^H (H Psi) is Hermitian: half of its tiles are computed, the rest mirrored
  rc = pwh_gram_herm(h->npw, nband, (const pwh_c128*)h->st_psi, h->npw, (const pwh_c128*)h->st_hpsi, h->npw,
                     (pwh_c128*)h->st_g, nband, h->st_ws, h->st_ws_bytes, st);
  if (rc) return rc;
  if (hpsi_host)
    CUDA_TRY(cudaMemcpy2DAsync(hpsi_host, (size_t)ldh * sizeof(c128), h->st_hpsi, row, row, nband, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaMemcpy2DAsync(G_host, (size_t)ldg * sizeof(c128), h->st_g, (size_t)nband * sizeof(c128),
                             (size_t)nband * sizeof(c128), nband, cudaMemcpyDeviceToHost, st));
  return PWH_OK;
}

extern "C" int pwh_sweep_host(pwh_ham* h, int64_t nband, int64_t block, pwh_c128* psi_host, int64_t ld, int degree,
                              double a, double b, double a0, pwh_c128* hpsi_host, int64_t ldh, pwh_c128* G_host,
                              int64_t ldg, void* stream) {
  if (!h) return fail(PWH_EINVAL, "handle is null");
  if (nband < 0) return fail(PWH_EINVAL, "nband < 0");
  if (degree < 0 || !(b > a) || !(a0 < a)) return fail(PWH_EINVAL, "bad filter parameters");
  if (nband == 0) return PWH_OK;
  if (!psi_host || !G_host) return fail(PWH_EINVAL, "null argument");
  if (ld < h->npw || ldg < nband || (hpsi_host && ldh < h->npw)) return fail(PWH_EINVAL, "leading dimension too small");
  cudaStream_t st = (cudaStream_t)stream;
  if (block <= 0 || block > nband) block = nband;
  return host_finish(h, st, sweep_host_impl(h, nband, block, psi_host, ld, degree, a, b, a0, hpsi_host, ldh, G_host, ldg, st));
}

extern "C" int pwh_probe_fp64_tensor_peak(int iters, double* tflops, void* stream) {
  if (!tflops || iters < 1) return fail(PWH_EINVAL, "bad arguments");
  double* sink = nullptr;
  CUDA_TRY(cudaMalloc(&sink, 16));
  const int ctas = 148 * 2;
  float ms = 0.f;
  cudaError_t e = dmma_probe(iters, ctas, sink, (cudaStream_t)stream, &ms);
  cudaFree(sink);
  CUDA_TRY(e);
  *tflops = (double)ctas * 8.0 * (double)iters * 32.0 * 512.0 / ((double)ms * 1e-3) * 1e-12;
  return PWH_OK;
}

extern "C" int pwh_profile_begin(void) {
  std::lock_guard<std::mutex> lk(g_prof_mu);
  for (auto& r : g_prof) { g_prof_pool.push_back(r.e0); g_prof_pool.push_back(r.e1); }
  g_prof.clear();
  g_prof_on.store(true);
  return PWH_OK;
}

extern "C" int pwh_profile_end(double ms[PWH_NSTAGES], int64_t launches[PWH_NSTAGES]) {
  if (!ms || !launches) return fail(PWH_EINVAL, "null argument");
  g_prof_on.store(false);
  const cudaError_t esync = cudaDeviceSynchronize();
  std::lock_guard<std::mutex> lk(g_prof_mu);
  if (esync != cudaSuccess) {
    for (auto& r : g_prof) { g_prof_pool.push_back(r.e0); g_prof_pool.push_back(r.e1); }
    g_prof.clear();
    return fail(PWH_ECUDA, "cudaDeviceSynchronize: %s", cudaGetErrorString(esync));
  }
  for (int i = 0; i < PWH_NSTAGES; ++i) { ms[i] = 0.0; launches[i] = 0; }
  cudaError_t first = cudaSuccess;
  for (auto& r : g_prof) {
    float t = 0.f;
    const cudaError_t e = cudaEventElapsedTime(&t, r.e0, r.e1);
    if (e != cudaSuccess && first == cudaSuccess) first = e;
    if (e == cudaSuccess && r.stage >= 0 && r.stage < PWH_NSTAGES) { ms[r.stage] += (double)t; launches[r.stage] += 1; }
    g_prof_pool.push_back(r.e0);
    g_prof_pool.push_back(r.e1);
  }
  g_prof.clear();
  if (first != cudaSuccess) return fail(PWH_ECUDA, "cudaEventElapsedTime: %s", cudaGetErrorString(first));
  return PWH_OK;
}

extern "C" int64_t pwh_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

extern "C" const char* pwh_last_error(void) { return g_err.c_str(); }
