// rwgt_api.cu — C ABI of include/rwgt.h: handle management, parameter preparation, kernel dispatch.
#include <cuda_runtime.h>
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/rwgt.h"
#include "kernels_small.cuh"
#include "bg_engine.cuh"
#include "photon_kernel.cuh"
#include "qq_kernels.cuh"
#include "event_file.cuh"

namespace {

thread_local char g_err[512] = "";
void set_err(const char* fmt, const char* a = "") { std::snprintf(g_err, sizeof(g_err), fmt, a); }

enum Proc { P_EPEM = 0, P_GG_TTX = 1, P_BG = 2, P_PHOTONS = 3, P_QQ = 4, P_MULTI = 5 };
const double PI = 3.14159265358979323846;

// A handle's tables and kernel attributes live on the device that was current at rwgt_create: every call that launches or
// copies makes that device current for its duration and restores the caller's device afterwards.
struct DeviceGuard {
  int prev = -1; bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    if (prev == dev) prev = -1;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

// ---------------------------------------------------------------------------- scratch of rwgt_sum_weights_static
// For callers that may not allocate (include/rwgt.h): the block partials and row counters of the eq. 2 reduction in a fixed array of
// the library image instead of a handle's cudaMalloc'ed buffers.  Layout: double partial[17][SUM_BLOCKS] at byte 0 (8,704 bytes),
// unsigned ticket[17] at byte 8,704.  One copy per GPU that loads the library; shared by every call on that GPU.
static_assert(RWGT_STATIC_SUM_MAX_ROWS == 1 + RWGT_MAX_SETS, "one call sums the old weights and every parameter set");
constexpr size_t STATIC_TICKET_OFFSET = sizeof(double) * RWGT_STATIC_SUM_MAX_ROWS * rwgt::SUM_BLOCKS;
static_assert(STATIC_TICKET_OFFSET % 256 == 0 && STATIC_TICKET_OFFSET + sizeof(unsigned) * RWGT_STATIC_SUM_MAX_ROWS <= RWGT_STATIC_SCRATCH_BYTES, "static scratch layout");
static __device__ __align__(256) unsigned char g_static_scratch[RWGT_STATIC_SCRATCH_BYTES];

namespace {
// In host code `g_static_scratch` names a host-side shadow of the array, not memory a kernel can use: the address a kernel may be
// given comes from cudaGetSymbolAddress, asked once per device with that device current, and is kept here.
std::mutex g_static_mutex;
unsigned char* g_static_ptr[RWGT_STATIC_MAX_DEVICES] = {};

// device address of the static scratch on the CURRENT device (looked up on the first call per device); nullptr + rc on failure
unsigned char* static_scratch_of_current_device(int* rc) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { set_err("rwgt_sum_weights_static: %s", cudaGetErrorString(e)); *rc = (int)e; return nullptr; }
  if (dev < 0 || dev >= RWGT_STATIC_MAX_DEVICES) { set_err("rwgt_sum_weights_static: device ordinal beyond RWGT_STATIC_MAX_DEVICES"); *rc = -1; return nullptr; }
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p) {
      set_err("rwgt_sum_weights_static: cudaGetSymbolAddress: %s", e != cudaSuccess ? cudaGetErrorString(e) : "null address");
      *rc = e != cudaSuccess ? (int)e : -1; return nullptr;
    }
    g_static_ptr[dev] = (unsigned char*)p;
  }
  *rc = 0;
  return g_static_ptr[dev];
}
}  // namespace

#define RWGT_MAX_CHUNKS 8
struct rwgt_handle {
  int proc;
  int n_ext;
  int n_gluons;
  int precision;
  int device;
  int nsets;                  // 1 + K
  rwgt_params sets[1 + RWGT_MAX_SETS];   // [0] = old, [1..K] = new
  rwgt::EpemParams epem;
  rwgt::GGttxParams ggttx;
  rwgt::PhotonParams photons; // e+ e- -> n_photons gamma
  int n_photons, sm_count;
  rwgt::QQParams qq;          // q qbar -> t tbar (+ g); n_gluons = number of radiated gluons
  int nsub;                   // P_MULTI ("LO multiprocess"): sub-handles, one per process of the mixed event list
  rwgt_handle* sub[RWGT_MAX_PROCESSES];
  int* d_idx; int* h_idx; long long idx_cap;     // per-process event index lists (device, pinned host), grown on demand
  rwgt::BgProcess* bg;        // ordered-current engine (n_gluons >= 3, or gg_ttx when forced)
  // device scratch for rwgt_run_host
  double* scratch;
  size_t scratch_bytes;
  char process[32];           // the process name as given to rwgt_create (without any "@" suffix); checked against event files
  double* sum_partial; unsigned* sum_ticket; double* sum_out;      // device scratch of rwgt_sum_weights (eq. 2), allocated at create
  rwgt::FileBuffers fb;       // pinned double buffers of rwgt_run_file (allocated on first use)
  int pipe_ready;                                     // copy streams and events below exist (all of them or none)
  cudaStream_t s_in, s_out;                           // copy streams of rwgt_run_host (created on first use)
  cudaEvent_t ev_in[RWGT_MAX_CHUNKS + 1], ev_k[RWGT_MAX_CHUNKS + 1];
};

static bool valid_params(const rwgt_params* p) {
  if (!p) return false;
  if (!(p->alpha_em > 0) || !(p->alpha_s > 0)) return false;
  if (!(p->sin2_thetaW > 0 && p->sin2_thetaW < 1)) return false;
  if (!(p->mZ > 0) || !(p->GammaZ >= 0) || !(p->mt >= 0)) return false;
  if (p->Gamma_t != 0.0) return false;
  if (!std::isfinite(p->ggg_scale) || !std::isfinite(p->gggg_scale)) return false;
  return true;
}

static rwgt::EpemSet make_epem(const rwgt_params& p) {
  rwgt::EpemSet s;
  s.e2 = 4.0 * PI * p.alpha_em;
  s.gz2 = s.e2 / (p.sin2_thetaW * (1.0 - p.sin2_thetaW));
  s.gL = -0.5 + p.sin2_thetaW;
  s.gR = p.sin2_thetaW;
  s.mZ2 = p.mZ * p.mZ;
  s.mZGZ = p.mZ * p.GammaZ;
  return s;
}

// device scratch every handle owns from the start (nothing is allocated inside rwgt_run / rwgt_sum_weights)
static rwgt_handle* finish_create(rwgt_handle* h) {
  const int rows = 1 + RWGT_MAX_SETS;
  cudaError_t e = cudaMalloc((void**)&h->sum_partial, sizeof(double) * rows * rwgt::SUM_BLOCKS);
  if (e == cudaSuccess) e = cudaMalloc((void**)&h->sum_ticket, sizeof(unsigned) * rows);
  if (e == cudaSuccess) e = cudaMalloc((void**)&h->sum_out, sizeof(double) * rows);
  if (e == cudaSuccess) e = cudaMemset(h->sum_ticket, 0, sizeof(unsigned) * rows);
  if (e != cudaSuccess) { set_err("rwgt_create: %s", cudaGetErrorString(e)); rwgt_destroy(h); return nullptr; }
  return h;
}

extern "C" {

const char* rwgt_last_error(void) { return g_err; }

#ifndef RWGT_BUILD_ID
#define RWGT_BUILD_ID "unknown"
#endif
const char* rwgt_build_id(void) { return RWGT_BUILD_ID; }

rwgt_handle* rwgt_create_multi(const char* process, const rwgt_params* params_old, const rwgt_params* params_new, int n_new) {
  if (!process || !params_old || !params_new) { set_err("rwgt_create: NULL argument"); return nullptr; }
  if (n_new < 1 || n_new > RWGT_MAX_SETS) { set_err("rwgt_create: number of new parameter sets must be in 1..RWGT_MAX_SETS"); return nullptr; }
  bool okp = valid_params(params_old);
  for (int k = 0; k < n_new; k++) okp = okp && valid_params(params_new + k);
  if (!okp) { set_err("rwgt_create: invalid parameter set for %s", process); return nullptr; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); set_err("rwgt_create: no CUDA device (this library has no CPU path)"); return nullptr; }
  rwgt_handle* h = new (std::nothrow) rwgt_handle();
  if (!h) { set_err("rwgt_create: out of memory"); return nullptr; }
  h->proc = -1; h->precision = RWGT_FP64; h->bg = nullptr; h->scratch = nullptr; h->scratch_bytes = 0; h->s_in = nullptr; h->s_out = nullptr; h->pipe_ready = 0;
  h->sum_partial = nullptr; h->sum_ticket = nullptr; h->sum_out = nullptr;
  h->nsub = 0; h->d_idx = nullptr; h->h_idx = nullptr; h->idx_cap = 0;
  h->nsets = 1 + n_new; h->sets[0] = *params_old;
  for (int k = 0; k < n_new; k++) h->sets[1 + k] = params_new[k];
  cudaGetDevice(&h->device);
  { int sms = 0; cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->device); h->sm_count = sms > 0 ? sms : 1; }
  std::string p(process);
  // "@bg" suffix routes gg_ttx through the generic ordered-current engine (used by the tests to cross-check it)
  bool force_bg = false;
  if (p.size() > 3 && p.compare(p.size() - 3, 3, "@bg") == 0) { force_bg = true; p.resize(p.size() - 3); }
  std::memset(h->process, 0, sizeof(h->process)); std::strncpy(h->process, p.c_str(), sizeof(h->process) - 1);
  int ng = -1;
  if (p == "epem_mupmum") { h->proc = P_EPEM; h->n_ext = 4; h->n_gluons = 0; }
  else if (p == "gg_ttx") { ng = 2; }
  else if (p == "gg_ttxg") { ng = 3; }
  else if (p == "gg_ttxgg") { ng = 4; }
  else if (p == "gg_ttxggg") { ng = 5; }
  else if (p == "qqx_ttx" || p == "qqx_ttxg") {
    // q qbar -> t tbar (+ g): a structurally different amplitude for the final states of gg_ttx / gg_ttxg
    const int ngl = (p == "qqx_ttxg") ? 1 : 0;
    h->proc = P_QQ; h->n_gluons = ngl; h->n_ext = 4 + ngl; h->qq.nsets = h->nsets; h->qq.two_pass = 0;
    for (int k = 0; k < h->nsets; k++) {
      const double g2 = 4.0 * PI * h->sets[k].alpha_s;
      h->qq.mt[k] = h->sets[k].mt; h->qq.r[k] = h->sets[k].ggg_scale;
      h->qq.fac[k] = ngl ? 2.0 * g2 * g2 * g2 / 36.0 : 2.0 * 2.0 * g2 * g2 / 36.0;
      if (h->sets[k].mt != h->sets[0].mt) h->qq.two_pass = 1;
    }
    // colour matrix of the four structures C_1 = (T^a T^c)_ji T^c_kl, C_2 = (T^c T^a)_ji T^c_kl, C_3 = T^c_ji (T^a T^c)_kl,
    // C_4 = T^c_ji (T^c T^a)_kl: G_ab = Tr(L_a(c) L_b(d)^+) Tr(K_a(c) K_b(d)^+), exact integers over 6^3 (labels a = 0, c = 1, d = 2)
    for (int x = 0; x < 4; x++) for (int y = 0; y < 4; y++) {
      auto light = [](int s, int lab) { return s == 0 ? std::vector<int>{0, lab} : s == 1 ? std::vector<int>{lab, 0} : std::vector<int>{lab}; };
      auto top = [](int s, int lab) { return s == 2 ? std::vector<int>{0, lab} : s == 3 ? std::vector<int>{lab, 0} : std::vector<int>{lab}; };
      std::vector<int> wl = light(x, 1), rl = light(y, 2), wt = top(x, 1), rt = top(y, 2);
      wl.insert(wl.end(), rl.rbegin(), rl.rend()); wt.insert(wt.end(), rt.rbegin(), rt.rend());
      h->qq.G[4 * x + y] = (double)rwgt::fierz_reduce({wl, wt}) / 216.0;
    }
    return finish_create(h);
  }
  else if (p == "epem_aa" || p == "epem_aaa" || p == "epem_aaaa" || p == "epem_aaaaa") {
    // e+ e- -> n photons (n = 5: the paper's measured process): only alpha_em enters, as e^(2n)
    const int na = (int)p.size() - 5;
    h->proc = P_PHOTONS; h->n_photons = na; h->n_ext = na + 2; h->n_gluons = 0; h->photons.nsets = h->nsets;
    double fact = 1; for (int i = 2; i <= na; i++) fact *= i;
    for (int k = 0; k < h->nsets; k++) h->photons.fac[k] = 2.0 * std::pow(4.0 * PI * h->sets[k].alpha_em, na) / (4.0 * fact);
    cudaError_t e = rwgt::photon_prepare(na);
    if (e != cudaSuccess) { set_err("rwgt_create: %s", cudaGetErrorString(e)); delete h; return nullptr; }
    return finish_create(h);
  }
  else { set_err("rwgt_create: unknown process '%s'", process); delete h; return nullptr; }
  if (h->proc == P_EPEM) {
    h->epem.nsets = h->nsets;
    for (int k = 0; k < h->nsets; k++) h->epem.set[k] = make_epem(h->sets[k]);
    return finish_create(h);
  }
  h->n_gluons = ng; h->n_ext = ng + 2;
  if (ng == 2 && !force_bg) {
    h->proc = P_GG_TTX;
    h->ggttx.nsets = h->nsets; h->ggttx.two_pass = 0;
    for (int k = 0; k < h->nsets; k++) {
      double gs2 = 4.0 * PI * h->sets[k].alpha_s;
      h->ggttx.mt[k] = h->sets[k].mt; h->ggttx.fac[k] = gs2 * gs2 / 256.0; h->ggttx.s3[k] = h->sets[k].ggg_scale;
      if (h->sets[k].mt != h->sets[0].mt) h->ggttx.two_pass = 1;
    }
    return finish_create(h);
  }
  h->proc = P_BG;
  std::string err;
  h->bg = rwgt::bg_create(ng, h->sets, h->nsets, err);
  if (!h->bg) { set_err("rwgt_create: %s", err.c_str()); delete h; return nullptr; }
  return finish_create(h);
}

rwgt_handle* rwgt_create(const char* process, const rwgt_params* params_old, const rwgt_params* params_new) {
  return rwgt_create_multi(process, params_old, params_new, 1);
}

int rwgt_n_sets(const rwgt_handle* h) { return h ? h->nsets - 1 : -1; }

int rwgt_set_precision(rwgt_handle* h, int mode) {
  if (!h || mode < 0 || mode > 2) { set_err("rwgt_set_precision: bad argument"); return -1; }
  if (h->proc == P_MULTI) {            // applies to the members that have the mode; the others stay FP64
    int with_mode = 0;
    for (int i = 0; i < h->nsub; i++) with_mode += (h->sub[i]->proc == P_BG);
    if (mode != RWGT_FP64 && with_mode == 0) { set_err("rwgt_set_precision: every member process of this handle is FP64 only"); return -1; }
    for (int i = 0; i < h->nsub; i++) if (h->sub[i]->proc == P_BG) h->sub[i]->precision = mode;
    h->precision = mode; return 0;
  }
  if (h->proc != P_BG && mode != RWGT_FP64) { set_err("rwgt_set_precision: this process is FP64 only"); return -1; }
  h->precision = mode;
  return 0;
}

int rwgt_n_external(const rwgt_handle* h) { return h ? h->n_ext : -1; }

double rwgt_flops_per_event(const rwgt_handle* h) {
  if (!h) return -1.0;
  // the two one-event-per-thread kernels: executed counts (2 DFMA + DMUL + DADD thread instructions per event) of an ncu capture; the
  // current build's capture is in profiles/counts.json (408 and 2,935) and bench.py prints model / ncu beside the roofline, so a stale
  // constant shows
  if (h->proc == P_EPEM) return 408.0 + (h->nsets - 2) * 45.0;
  if (h->proc == P_PHOTONS) return rwgt::photon_flops_per_event(h->n_photons);
  // q qbar -> t tbar (g): operation count of qq_kernels.cuh (externals ~300; per gluon helicity b_1, b_2, l ~550; per (gluon, tbar) helicity five
  // slash chains ~700; per helicity 5 row.col ~130 + per set the 4 x 4 colour form ~70), calibrated to the executed count (the compiler folds the
  // zero components of eps and of the massless spinors): ncu 6,398 flops per event for two sets (profiles/counts.json, cfg8_fp64), 582 without the gluon
  if (h->proc == P_QQ) { const double one = h->n_gluons ? 300.0 + 2 * 550.0 + 4 * 700.0 + 8 * (130.0 + h->nsets * 70.0) : 300.0 + 2 * 64.0 + 4 * 36.0;
                         return h->qq.two_pass ? h->nsets * one : one; }
  if (h->proc == P_MULTI) { double f = 0; for (int i = 0; i < h->nsub; i++) f += rwgt_flops_per_event(h->sub[i]); return f / h->nsub; }
  // gg_ttx: 2902 for two sets of equal mass; a further set of equal mass costs 8 helicities x (4 FMA + colour form 5 FMA + 4 MUL/ADD)
  if (h->proc == P_GG_TTX) return h->ggttx.two_pass ? h->nsets * 2902.0 : 2902.0 + (h->nsets - 2) * 8 * 26.0;
  return rwgt::bg_flops_per_event(h->bg, h->precision);
}

double rwgt_tensor_flops_per_event(const rwgt_handle* h) {
  if (!h) return -1.0;
  if (h->proc == P_MULTI) { double f = 0; for (int i = 0; i < h->nsub; i++) f += rwgt_tensor_flops_per_event(h->sub[i]); return f / h->nsub; }
  return h->proc == P_BG ? rwgt::bg_tensor_flops_per_event(h->bg) : 0.0;
}

// one kernel launch over events [0, n) of buffers whose momentum planes are `stride` events apart and whose per-set
// output planes are `ostride` events apart
static int launch_events(rwgt_handle* h, const double* momenta, const double* weights, double* out_me_old, double* out_me_new,
                         double* out_w_new, long long n, long long stride, long long ostride, cudaStream_t st, const int* idx = nullptr) {
  if (idx && (h->proc == P_EPEM || h->proc == P_PHOTONS)) { set_err("rwgt_run: this process cannot be part of a multiprocess handle"); return -1; }
  if (h->proc == P_EPEM) {
    // small event sets (cfg 1 has 16,384): 64-thread CTAs, so that the grid covers all SMs (256 CTAs instead of 64 on 148 SMs)
    int bs = (n < 512LL * h->sm_count) ? 64 : rwgt::RWGT_EPEM_BS; long long nb = (n + bs - 1) / bs;
    rwgt::epem_mupmum_kernel<<<(unsigned)nb, bs, 0, st>>>(momenta, weights, out_me_old, out_me_new, out_w_new, n, stride, ostride, h->epem);
  } else if (h->proc == P_GG_TTX) {
    int bs = h->nsets == 2 ? rwgt::GGTTX_BS : 128; long long nb = (n + bs - 1) / bs;
    if (h->nsets == 2) rwgt::gg_ttx_kernel<<<(unsigned)nb, bs, 0, st>>>(momenta, weights, idx, out_me_old, out_me_new, out_w_new, n, stride, ostride, h->ggttx);
    else rwgt::gg_ttx_multi_kernel<<<(unsigned)nb, bs, 0, st>>>(momenta, weights, idx, out_me_old, out_me_new, out_w_new, n, stride, ostride, h->ggttx);
  } else if (h->proc == P_QQ) {
    int bs = 128; long long nb = (n + bs - 1) / bs;
    if (h->n_gluons) rwgt::qqx_ttx_kernel<1><<<(unsigned)nb, bs, 0, st>>>(momenta, weights, idx, out_me_old, out_me_new, out_w_new, n, stride, ostride, h->qq);
    else rwgt::qqx_ttx_kernel<0><<<(unsigned)nb, bs, 0, st>>>(momenta, weights, idx, out_me_old, out_me_new, out_w_new, n, stride, ostride, h->qq);
  } else if (h->proc == P_PHOTONS) {
    cudaError_t e = rwgt::photon_launch(h->n_photons, h->sm_count, st, momenta, weights, out_me_old, out_me_new, out_w_new, n, stride, ostride, h->photons);
    if (e != cudaSuccess) { set_err("rwgt_run: %s", cudaGetErrorString(e)); return (int)e; }
  } else {
    int rc = rwgt::bg_run(h->bg, h->precision, momenta, weights, idx, out_me_old, out_me_new, out_w_new, n, stride, ostride, st);
    if (rc != 0) { set_err("rwgt_run: engine launch failed"); return rc; }
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_err("rwgt_run: %s", cudaGetErrorString(e)); return (int)e; }
  return 0;
}

int rwgt_run_multi(rwgt_handle* h, const double* momenta, const double* weights, double* out_me_old, double* out_me_new,
                   double* out_w_new, long long n_events, void* stream) {
  if (!h || n_events < 0) { set_err("rwgt_run: bad handle or n_events < 0"); return -1; }
  if (n_events == 0) return 0;
  if (!momenta || !weights || !out_me_old || !out_me_new || !out_w_new) { set_err("rwgt_run: NULL buffer"); return -1; }
  if (h->proc == P_MULTI) { set_err("rwgt_run: multiprocess handle, use rwgt_run_multiprocess"); return -1; }
  DeviceGuard guard(h->device);
  if (!guard.ok) { set_err("rwgt_run: cannot make the handle's device current"); return -1; }
  return launch_events(h, momenta, weights, out_me_old, out_me_new, out_w_new, n_events, n_events, n_events, (cudaStream_t)stream);
}

int rwgt_run(rwgt_handle* h, const double* momenta, const double* weights, double* out_me_old, double* out_me_new,
             double* out_w_new, long long n_events, void* stream) {
  if (h && h->nsets != 2) { set_err("rwgt_run: handle has several new parameter sets, use rwgt_run_multi"); return -1; }
  return rwgt_run_multi(h, momenta, weights, out_me_old, out_me_new, out_w_new, n_events, stream);
}

// Host-buffer path (the transfers are part of what a user pays).  The events are cut into chunks; the
// host->device copy of chunk c+1 (copy stream), the kernel of chunk c (caller's stream) and the device->host copy of
// chunk c-1 (second copy stream) overlap, so on a full-duplex link the call costs about max(H2D, D2H, kernel).
int rwgt_run_multi_host(rwgt_handle* h, const double* momenta, const double* weights, double* out_me_old, double* out_me_new,
                        double* out_w_new, long long n_events, void* stream) {
  if (!h || n_events < 0) { set_err("rwgt_run_host: bad handle or n_events < 0"); return -1; }
  if (n_events == 0) return 0;
  if (!momenta || !weights || !out_me_old || !out_me_new || !out_w_new) { set_err("rwgt_run_host: NULL buffer"); return -1; }
  if (h->proc == P_MULTI) { set_err("rwgt_run_host: multiprocess handle, use rwgt_run_multiprocess"); return -1; }
  DeviceGuard guard(h->device);
  if (!guard.ok) { set_err("rwgt_run_host: cannot make the handle's device current"); return -1; }
  cudaStream_t st = (cudaStream_t)stream;
  const size_t n = (size_t)n_events, planes = (size_t)h->n_ext * 4, nin = planes * n, K = (size_t)h->nsets - 1, need = (nin + (2 + 2 * K) * n) * sizeof(double);
  cudaError_t e = cudaSuccess;
  if (need > h->scratch_bytes) {
    if (h->scratch) cudaFree(h->scratch);
    h->scratch = nullptr; h->scratch_bytes = 0;
    e = cudaMalloc((void**)&h->scratch, need);
    if (e != cudaSuccess) { h->scratch = nullptr; set_err("rwgt_run_host: %s", cudaGetErrorString(e)); return (int)e; }
    h->scratch_bytes = need;
  }
  if (!h->pipe_ready) {
    // copy streams and events: all or nothing
    cudaStream_t si = nullptr, so = nullptr; cudaEvent_t ei[RWGT_MAX_CHUNKS + 1] = {}, ek[RWGT_MAX_CHUNKS + 1] = {};
    e = cudaStreamCreateWithFlags(&si, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&so, cudaStreamNonBlocking);
    for (int c = 0; c <= RWGT_MAX_CHUNKS && e == cudaSuccess; c++) {
      e = cudaEventCreateWithFlags(&ei[c], cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ek[c], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) {
      for (int c = 0; c <= RWGT_MAX_CHUNKS; c++) { if (ei[c]) cudaEventDestroy(ei[c]); if (ek[c]) cudaEventDestroy(ek[c]); }
      if (si) cudaStreamDestroy(si); if (so) cudaStreamDestroy(so);
      set_err("rwgt_run_host: %s", cudaGetErrorString(e)); return (int)e;
    }
    h->s_in = si; h->s_out = so;
    for (int c = 0; c <= RWGT_MAX_CHUNKS; c++) { h->ev_in[c] = ei[c]; h->ev_k[c] = ek[c]; }
    h->pipe_ready = 1;
  }
  double* d_mom = h->scratch; double* d_w = d_mom + nin; double* d_a = d_w + n; double* d_b = d_a + n; double* d_o = d_b + K * n;
  // chunks of >= 64 Ki events, at most RWGT_MAX_CHUNKS
  long long nchunk = (long long)((n + 65535) / 65536); if (nchunk > RWGT_MAX_CHUNKS) nchunk = RWGT_MAX_CHUNKS; if (nchunk < 1) nchunk = 1;
  long long per = ((long long)n + nchunk - 1) / nchunk;
  int rc = 0;
  // on any error: stop issuing, then drain the three streams so that no copy is still touching the caller's buffers on return
#define RWGT_CK(call) do { if (rc == 0) { e = (call); if (e != cudaSuccess) { set_err("rwgt_run_host: %s", cudaGetErrorString(e)); rc = (int)e; } } } while (0)
  // the scratch may still be in use by earlier work on the caller's stream
  RWGT_CK(cudaEventRecord(h->ev_in[RWGT_MAX_CHUNKS], st));
  RWGT_CK(cudaStreamWaitEvent(h->s_in, h->ev_in[RWGT_MAX_CHUNKS], 0));
  for (long long c = 0; c < nchunk && rc == 0; c++) {
    long long a0 = c * per, cnt = std::min<long long>(per, (long long)n - a0);
    if (cnt <= 0) break;
    RWGT_CK(cudaMemcpy2DAsync(d_mom + a0, n * sizeof(double), momenta + a0, n * sizeof(double), (size_t)cnt * sizeof(double), planes,
                              cudaMemcpyHostToDevice, h->s_in));
    RWGT_CK(cudaMemcpyAsync(d_w + a0, weights + a0, (size_t)cnt * sizeof(double), cudaMemcpyHostToDevice, h->s_in));
    RWGT_CK(cudaEventRecord(h->ev_in[c], h->s_in));
    RWGT_CK(cudaStreamWaitEvent(st, h->ev_in[c], 0));
    if (rc == 0) rc = launch_events(h, d_mom + a0, d_w + a0, d_a + a0, d_b + a0, d_o + a0, cnt, (long long)n, (long long)n, st);
    RWGT_CK(cudaEventRecord(h->ev_k[c], st));
    RWGT_CK(cudaStreamWaitEvent(h->s_out, h->ev_k[c], 0));
    RWGT_CK(cudaMemcpyAsync(out_me_old + a0, d_a + a0, (size_t)cnt * sizeof(double), cudaMemcpyDeviceToHost, h->s_out));
    RWGT_CK(cudaMemcpy2DAsync(out_me_new + a0, n * sizeof(double), d_b + a0, n * sizeof(double), (size_t)cnt * sizeof(double), K, cudaMemcpyDeviceToHost, h->s_out));
    RWGT_CK(cudaMemcpy2DAsync(out_w_new + a0, n * sizeof(double), d_o + a0, n * sizeof(double), (size_t)cnt * sizeof(double), K, cudaMemcpyDeviceToHost, h->s_out));
  }
  // the caller's stream continues only after the results are on the host; then wait for it
  RWGT_CK(cudaEventRecord(h->ev_k[RWGT_MAX_CHUNKS], h->s_out));
  RWGT_CK(cudaStreamWaitEvent(st, h->ev_k[RWGT_MAX_CHUNKS], 0));
  RWGT_CK(cudaStreamSynchronize(st));
#undef RWGT_CK
  if (rc != 0) { cudaStreamSynchronize(h->s_in); cudaStreamSynchronize(st); cudaStreamSynchronize(h->s_out); }
  return rc;
}

int rwgt_run_host(rwgt_handle* h, const double* momenta, const double* weights, double* out_me_old, double* out_me_new,
                  double* out_w_new, long long n_events, void* stream) {
  if (h && h->nsets != 2) { set_err("rwgt_run_host: handle has several new parameter sets, use rwgt_run_multi_host"); return -1; }
  return rwgt_run_multi_host(h, momenta, weights, out_me_old, out_me_new, out_w_new, n_events, stream);
}

// real-emission contributions "can be treated as LO multiprocesses" -- one event list, several amplitudes
rwgt_handle* rwgt_create_multiprocess(const char* processes, const rwgt_params* params_old, const rwgt_params* params_new, int n_new) {
  if (!processes || !params_old || !params_new) { set_err("rwgt_create_multiprocess: NULL argument"); return nullptr; }
  std::vector<std::string> names; { std::string all(processes), cur; for (char ch : all) { if (ch == ',') { names.push_back(cur); cur.clear(); } else if (ch != ' ') cur += ch; } names.push_back(cur); }
  if (names.empty() || (int)names.size() > RWGT_MAX_PROCESSES) { set_err("rwgt_create_multiprocess: 1..RWGT_MAX_PROCESSES comma-separated process names"); return nullptr; }
  rwgt_handle* h = new (std::nothrow) rwgt_handle();
  if (!h) { set_err("rwgt_create_multiprocess: out of memory"); return nullptr; }
  h->proc = P_MULTI; h->precision = RWGT_FP64; h->bg = nullptr; h->scratch = nullptr; h->scratch_bytes = 0; h->s_in = nullptr; h->s_out = nullptr; h->pipe_ready = 0;
  h->sum_partial = nullptr; h->sum_ticket = nullptr; h->sum_out = nullptr; h->nsub = 0; h->d_idx = nullptr; h->h_idx = nullptr; h->idx_cap = 0;
  h->nsets = 1 + n_new; h->n_gluons = 0; h->n_ext = -1; std::memset(h->process, 0, sizeof(h->process));
  cudaGetDevice(&h->device);
  for (const std::string& nm : names) {
    rwgt_handle* s = rwgt_create_multi(nm.c_str(), params_old, params_new, n_new);       // sets g_err on failure
    if (s && (s->proc == P_EPEM || s->proc == P_PHOTONS)) { rwgt_destroy(s); s = nullptr; set_err("rwgt_create_multiprocess: '%s' cannot be a member (QCD processes only)", nm.c_str()); }
    if (s && h->n_ext >= 0 && s->n_ext != h->n_ext) { rwgt_destroy(s); s = nullptr; set_err("rwgt_create_multiprocess: '%s' has another number of external legs than the first process", nm.c_str()); }
    if (!s) { rwgt_destroy(h); return nullptr; }
    h->n_ext = s->n_ext; h->sub[h->nsub++] = s;
  }
  for (int k = 0; k < h->nsets; k++) h->sets[k] = h->sub[0]->sets[k];
  std::strncpy(h->process, "multiprocess", sizeof(h->process) - 1);
  return finish_create(h);
}

int rwgt_n_processes(const rwgt_handle* h) { return !h ? -1 : (h->proc == P_MULTI ? h->nsub : 1); }

int rwgt_run_multiprocess(rwgt_handle* h, const double* momenta, const double* weights, const int* process_id, double* out_me_old,
                          double* out_me_new, double* out_w_new, long long n_events, void* stream) {
  if (!h || h->proc != P_MULTI || n_events < 0) { set_err("rwgt_run_multiprocess: not a multiprocess handle, or n_events < 0"); return -1; }
  if (n_events == 0) return 0;
  if (!momenta || !weights || !process_id || !out_me_old || !out_me_new || !out_w_new) { set_err("rwgt_run_multiprocess: NULL buffer"); return -1; }
  if (n_events > 0x7fffffffLL) { set_err("rwgt_run_multiprocess: more than 2^31-1 events in one call"); return -1; }
  DeviceGuard guard(h->device);
  if (!guard.ok) { set_err("rwgt_run_multiprocess: cannot make the handle's device current"); return -1; }
  cudaStream_t st = (cudaStream_t)stream; cudaError_t e = cudaSuccess;
  if (n_events > h->idx_cap) {
    // the pinned list may still be the source of a copy enqueued by an earlier call
    if (h->h_idx) { cudaStreamSynchronize(st); cudaFreeHost(h->h_idx); h->h_idx = nullptr; }
    if (h->d_idx) { cudaFree(h->d_idx); h->d_idx = nullptr; }
    h->idx_cap = 0;
    e = cudaMalloc((void**)&h->d_idx, sizeof(int) * (size_t)n_events);
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&h->h_idx, sizeof(int) * (size_t)n_events, cudaHostAllocDefault);
    if (e != cudaSuccess) { set_err("rwgt_run_multiprocess: %s", cudaGetErrorString(e)); return (int)e; }
    h->idx_cap = n_events;
  } else cudaStreamSynchronize(st);               // an earlier call's copy out of h_idx must have finished before it is rewritten
  // stable partition of the event indices by process (host; 4 bytes per event against >= 136 bytes of momenta)
  long long count[RWGT_MAX_PROCESSES] = {}, off[RWGT_MAX_PROCESSES + 1] = {};
  for (long long i = 0; i < n_events; i++) { const int pid = process_id[i]; if (pid < 0 || pid >= h->nsub) { set_err("rwgt_run_multiprocess: process_id outside 0..n_processes-1"); return -1; } count[pid]++; }
  for (int k = 0; k < h->nsub; k++) off[k + 1] = off[k] + count[k];
  { long long fill[RWGT_MAX_PROCESSES]; for (int k = 0; k < h->nsub; k++) fill[k] = off[k];
    for (long long i = 0; i < n_events; i++) h->h_idx[fill[process_id[i]]++] = (int)i; }
  e = cudaMemcpyAsync(h->d_idx, h->h_idx, sizeof(int) * (size_t)n_events, cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) { set_err("rwgt_run_multiprocess: %s", cudaGetErrorString(e)); return (int)e; }
  for (int k = 0; k < h->nsub; k++) {
    if (count[k] == 0) continue;
    int rc = launch_events(h->sub[k], momenta, weights, out_me_old, out_me_new, out_w_new, count[k], n_events, n_events, st, h->d_idx + off[k]);
    if (rc != 0) return rc;
  }
  return 0;
}

// eq. 2: sigma ~ sum_k W_k, one deterministic device reduction per row
int rwgt_sum_weights(rwgt_handle* h, const double* w, int n_rows, long long n_events, double* out_sums, void* stream) {
  if (!h || n_events < 0 || n_rows < 1 || n_rows > 1 + RWGT_MAX_SETS) { set_err("rwgt_sum_weights: bad handle, n_events < 0 or n_rows outside 1..1+RWGT_MAX_SETS"); return -1; }
  if (!w || !out_sums) { set_err("rwgt_sum_weights: NULL buffer"); return -1; }
  DeviceGuard guard(h->device);
  if (!guard.ok) { set_err("rwgt_sum_weights: cannot make the handle's device current"); return -1; }
  rwgt::sum_rows_kernel<<<dim3(rwgt::SUM_BLOCKS, n_rows), rwgt::SUM_THREADS, 0, (cudaStream_t)stream>>>(w, n_events, n_events, h->sum_partial, h->sum_ticket, out_sums);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_err("rwgt_sum_weights: %s", cudaGetErrorString(e)); return (int)e; }
  return 0;
}

// eq. 2 without a handle and without any allocation (include/rwgt.h): the kernel of rwgt_sum_weights on the library's static scratch
int rwgt_sum_weights_static(const double* w, int n_rows, long long n_events, double* out_sums, void* stream) {
  if (n_rows < 1 || n_rows > RWGT_STATIC_SUM_MAX_ROWS) {
    set_err("rwgt_sum_weights_static: n_rows outside 1..RWGT_STATIC_SUM_MAX_ROWS (17): the static scratch holds 17 rows, sum the rest in a further call");
    return -1;
  }
  if (n_events < 0) { set_err("rwgt_sum_weights_static: n_events < 0"); return -1; }
  if (!w || !out_sums) { set_err("rwgt_sum_weights_static: NULL buffer"); return -1; }
  int rc = 0;
  unsigned char* base = static_scratch_of_current_device(&rc);
  if (!base) return rc;
  double* partial = (double*)base;
  unsigned* ticket = (unsigned*)(base + STATIC_TICKET_OFFSET);
  // the counters must start at zero whatever an earlier (possibly failed) call left behind; the partials are overwritten before use
  cudaError_t e = cudaMemsetAsync(ticket, 0, sizeof(unsigned) * RWGT_STATIC_SUM_MAX_ROWS, (cudaStream_t)stream);
  if (e != cudaSuccess) { set_err("rwgt_sum_weights_static: %s", cudaGetErrorString(e)); return (int)e; }
  rwgt::sum_rows_kernel<<<dim3(rwgt::SUM_BLOCKS, n_rows), rwgt::SUM_THREADS, 0, (cudaStream_t)stream>>>(w, n_events, n_events, partial, ticket, out_sums);
  e = cudaGetLastError();
  if (e != cudaSuccess) { set_err("rwgt_sum_weights_static: %s", cudaGetErrorString(e)); return (int)e; }
  return 0;
}

// PAPER.md:87 steps 2-8 on a binary SoA event file (csrc/event_file.cuh): read -> H2D -> kernel -> D2H -> write, pipelined
int rwgt_run_file(rwgt_handle* h, const char* in_path, const char* out_path, long long first_event, long long n_events, void* stream) {
  if (!h || !in_path || !out_path || first_event < 0) { set_err("rwgt_run_file: bad argument"); return -1; }
  DeviceGuard guard(h->device);
  if (!guard.ok) { set_err("rwgt_run_file: cannot make the handle's device current"); return -1; }
  int fin = ::open(in_path, O_RDONLY);
  if (fin < 0) { set_err("rwgt_run_file: cannot open %s", in_path); return -1; }
  rwgt_event_file_header hd;
  if (!rwgt::pread_all(fin, &hd, sizeof(hd), 0) || std::memcmp(hd.magic, "RWGTEVT1", 8) != 0 || hd.version != 1) { ::close(fin); set_err("rwgt_run_file: %s is not an event file (magic/version)", in_path); return -1; }
  if ((int)hd.n_ext != h->n_ext || std::strncmp(hd.process, h->process, sizeof(hd.process)) != 0) { ::close(fin); set_err("rwgt_run_file: %s holds events of another process", in_path); return -1; }
  struct stat sb;
  const long long planes = (long long)h->n_ext * 4, K = h->nsets - 1;
  // n_events comes from the file: bound it by the file's size BEFORE multiplying (a huge value must not wrap the product)
  if (::fstat(fin, &sb) != 0 || (long long)sb.st_size < (long long)sizeof(hd) ||
      hd.n_events > (unsigned long long)(((long long)sb.st_size - (long long)sizeof(hd)) / 8) / (unsigned long long)(planes + 1)) {
    ::close(fin); set_err("rwgt_run_file: %s is truncated", in_path); return -1;
  }
  const long long ntot = (long long)hd.n_events;
  if (n_events < 0) n_events = ntot - first_event;
  if (n_events < 0 || first_event > ntot || n_events > ntot - first_event) { ::close(fin); set_err("rwgt_run_file: event range outside the file"); return -1; }
  // the result goes to "<out_path>.tmp" and takes its name only when it is complete: a failed call leaves no well-formed result
  // file behind (and an existing out_path untouched); input and output must be different files
  struct stat so;
  if (::stat(out_path, &so) == 0 && so.st_dev == sb.st_dev && so.st_ino == sb.st_ino) { ::close(fin); set_err("rwgt_run_file: %s is the event file itself", out_path); return -1; }
  const std::string tmp_path = std::string(out_path) + ".tmp";
  if (::stat(tmp_path.c_str(), &so) == 0 && so.st_dev == sb.st_dev && so.st_ino == sb.st_ino) { ::close(fin); set_err("rwgt_run_file: %s.tmp is the event file itself", out_path); return -1; }
  int fout = ::open(tmp_path.c_str(), O_CREAT | O_TRUNC | O_RDWR, 0644);
  if (fout < 0) { ::close(fin); set_err("rwgt_run_file: cannot create %s.tmp", out_path); return -1; }
  rwgt_result_file_header ho; std::memset(&ho, 0, sizeof(ho));
  std::memcpy(ho.magic, "RWGTRES1", 8); ho.version = 1; ho.n_sets = (uint32_t)K; ho.n_events = (uint64_t)n_events; std::memcpy(ho.process, h->process, sizeof(ho.process));
  ho.first_event = (uint64_t)first_event;
  const long long n = n_events; const off_t obase = sizeof(ho);
  bool io_ok = rwgt::pwrite_all(fout, &ho, sizeof(ho), 0) && ::ftruncate(fout, obase + (off_t)((1 + 2 * K) * n + 1 + K) * 8) == 0;
  int rc = io_ok ? 0 : -1;
  if (!io_ok) set_err("rwgt_run_file: cannot write %s", out_path);
  double sums[1 + RWGT_MAX_SETS]; for (int k = 0; k <= K; k++) sums[k] = 0.0;
  if (rc == 0 && n > 0) {
    long long chunk = (n + 7) / 8; if (chunk < 16384) chunk = 16384; if (chunk > (1 << 19)) chunk = 1 << 19; if (chunk > n) chunk = n;
    chunk = (chunk + 1023) / 1024 * 1024;
    cudaError_t e = h->fb.ensure(chunk, (int)planes, (int)K);
    if (e != cudaSuccess) { set_err("rwgt_run_file: %s", cudaGetErrorString(e)); rc = (int)e; }
    const long long nchunk = (n + chunk - 1) / chunk;
    // reader: the chunk's planes (ntot apart in the file) into compact planes (cnt apart) of pinned buffer b
    auto read_chunk = [&](long long c, int b, bool* ok) {
      const long long a0 = c * chunk, cnt = std::min(chunk, n - a0); bool g = true;
      for (long long pl = 0; pl <= planes && g; pl++)
        g = rwgt::pread_all(fin, h->fb.in[b] + pl * cnt, (size_t)cnt * 8, (off_t)sizeof(hd) + (off_t)(pl * ntot + first_event + a0) * 8);
      *ok = g;
    };
    // writer: me_old | me_new[K] | w_new[K] rows (cnt apart in the buffer, n apart in the file)
    auto write_chunk = [&](long long c, int b, bool* ok) {
      const long long a0 = c * chunk, cnt = std::min(chunk, n - a0); bool g = true;
      for (long long r = 0; r < 1 + 2 * K && g; r++) g = rwgt::pwrite_all(fout, h->fb.out[b] + r * cnt, (size_t)cnt * 8, obase + (off_t)(r * n + a0) * 8);
      *ok = g;
    };
    bool rd_ok = true, wr_ok = true;
    std::thread reader, writer;
    if (rc == 0) reader = std::thread(read_chunk, 0LL, 0, &rd_ok);
    for (long long c = 0; c < nchunk && rc == 0; c++) {
      const int b = (int)(c & 1); const long long a0 = c * chunk, cnt = std::min(chunk, n - a0);
      reader.join();
      if (!rd_ok) { set_err("rwgt_run_file: read error on %s", in_path); rc = -1; break; }
      if (c + 1 < nchunk) reader = std::thread(read_chunk, c + 1, b ^ 1, &rd_ok);
      double* hi = h->fb.in[b]; double* o = h->fb.out[b];
      rc = rwgt_run_multi_host(h, hi, hi + planes * cnt, o, o + cnt, o + (1 + K) * cnt, cnt, stream);
      if (rc == 0) {
        // eq. 2 on the chunk while it is still in the device scratch (layout of rwgt_run_multi_host): sum W, sum W'_k
        const size_t nin = (size_t)planes * cnt; double* d_w = h->scratch + nin; double* d_o = d_w + (2 + K) * cnt;
        rc = rwgt_sum_weights(h, d_w, 1, cnt, h->sum_out, stream);
        if (rc == 0) rc = rwgt_sum_weights(h, d_o, (int)K, cnt, h->sum_out + 1, stream);
        double part[1 + RWGT_MAX_SETS];
        if (rc == 0) { e = cudaMemcpyAsync(part, h->sum_out, sizeof(double) * (1 + K), cudaMemcpyDeviceToHost, (cudaStream_t)stream);
                       if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
                       if (e != cudaSuccess) { set_err("rwgt_run_file: %s", cudaGetErrorString(e)); rc = (int)e; } }
        if (rc == 0) for (int k = 0; k <= K; k++) sums[k] += part[k];       // chunk order: deterministic for a given range
      }
      if (writer.joinable()) { writer.join(); if (!wr_ok) { set_err("rwgt_run_file: write error on %s", out_path); rc = -1; } }
      if (rc == 0) writer = std::thread(write_chunk, c, b, &wr_ok);
    }
    if (reader.joinable()) reader.join();
    if (writer.joinable()) { writer.join(); if (!wr_ok && rc == 0) { set_err("rwgt_run_file: write error on %s", out_path); rc = -1; } }
  }
  if (rc == 0 && !rwgt::pwrite_all(fout, sums, sizeof(double) * (1 + K), obase + (off_t)((1 + 2 * K) * n) * 8)) { set_err("rwgt_run_file: write error on %s", out_path); rc = -1; }
  ::close(fin);
  if (::close(fout) != 0 && rc == 0) { set_err("rwgt_run_file: write error on %s", out_path); rc = -1; }
  if (rc == 0 && ::rename(tmp_path.c_str(), out_path) != 0) { set_err("rwgt_run_file: cannot rename the finished result to %s", out_path); rc = -1; }
  if (rc != 0) ::unlink(tmp_path.c_str());
  return rc;
}

int rwgt_destroy(rwgt_handle* h) {
  if (!h) return -1;
  DeviceGuard guard(h->device);
  for (int i = 0; i < h->nsub; i++) rwgt_destroy(h->sub[i]);
  if (h->d_idx) cudaFree(h->d_idx);
  if (h->h_idx) cudaFreeHost(h->h_idx);
  if (h->bg) rwgt::bg_destroy(h->bg);
  if (h->scratch) cudaFree(h->scratch);
  cudaFree(h->sum_partial); cudaFree(h->sum_ticket); cudaFree(h->sum_out);
  h->fb.release();
  if (h->pipe_ready) {
    cudaStreamDestroy(h->s_in); cudaStreamDestroy(h->s_out);
    for (int c = 0; c <= RWGT_MAX_CHUNKS; c++) { cudaEventDestroy(h->ev_in[c]); cudaEventDestroy(h->ev_k[c]); }
  }
  delete h;
  return 0;
}

int rwgt_colour_matrix(int n_gluons, double* out) {
  if (n_gluons < 2 || n_gluons > 5 || !out) return -1;
  std::vector<double> C = rwgt::colour_matrix_fierz(n_gluons);
  std::memcpy(out, C.data(), C.size() * sizeof(double));
  int f = 1; for (int i = 2; i <= n_gluons; i++) f *= i;
  return f;
}

}  // extern "C"
