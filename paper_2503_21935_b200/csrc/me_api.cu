// me_api.cu -- the C ABI of include/me_b200.h: handles, tables, dispatch to the per-(process, precision)
// launchers of me_proc.cu.  Host code only; no kernel lives here.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <initializer_list>
#include <new>
#include <string>

#include "../../include/me_b200.h"
#include "me_kernels.cuh"
#include "me_rambo.h"

typedef int (*launch_fn)(const me::LaunchArgs&, int mode, void* stream, me::LaunchInfo* info, int dry);

#define ME_DECL(name)                                                                        \
  int me_launch_##name##_p0(const me::LaunchArgs&, int, void*, me::LaunchInfo*, int);        \
  int me_launch_##name##_p1(const me::LaunchArgs&, int, void*, me::LaunchInfo*, int);        \
  int me_launch_##name##_p2(const me::LaunchArgs&, int, void*, me::LaunchInfo*, int);
ME_DECL(ee_mumu)
ME_DECL(gg_tt)
ME_DECL(gg_ttg)
ME_DECL(gg_ttgg)
ME_DECL(gg_ttggg)
ME_DECL(gux_taptamux)
ME_DECL(gux_taptamgux)
ME_DECL(gux_taptamggux)

// multichannel (me_proc_diag.cu), gg processes only
typedef int (*diag_fn)(const me::LaunchArgs&, const int*, double*, double*, void*, void*);
typedef int (*chanflows_fn)(const unsigned**, int*);
typedef size_t (*diag_scratch_fn)();
#define ME_DECL_DIAG(name)                                                                          \
  int me_launch_diag_##name(const me::LaunchArgs&, const int*, double*, double*, void*, void*);    \
  int me_chanflows_##name(const unsigned**, int*);                                                  \
  size_t me_diag_scratch_##name();
ME_DECL_DIAG(gg_tt)
ME_DECL_DIAG(gg_ttg)
ME_DECL_DIAG(gg_ttgg)
ME_DECL_DIAG(gg_ttggg)

#include "gen/me_tables.h"

namespace {

struct ProcDesc {
  const char* name;
  int npar, ngl, ndiag;
  int denom;          // spin and colour average of the initial state x identical final-state particles
  int gluons[8];      // particle indices of the gluons
  int nmassive;       // the first nmassive final-state particles have the top mass (me_generate)
  launch_fn fn[3];
  diag_fn diag;
  chanflows_fn chanflows;
  diag_scratch_fn diag_scratch;
  const char* chan_keys;
};
#define ME_ROW(name, npar, ngl, ndiag, denom, ...) \
  { #name, npar, ngl, ndiag, denom, __VA_ARGS__, 2, { me_launch_##name##_p0, me_launch_##name##_p1, me_launch_##name##_p2 }, \
    me_launch_diag_##name, me_chanflows_##name, me_diag_scratch_##name, kChanKeys_##name }
const ProcDesc kProcs[] = {
    { "ee_mumu", 4, 0, 2, 4, {0}, 0, { me_launch_ee_mumu_p0, me_launch_ee_mumu_p1, me_launch_ee_mumu_p2 }, nullptr, nullptr, nullptr, kChanKeys_ee_mumu },
    ME_ROW(gg_tt, 4, 2, 3, 256, {0, 1}), ME_ROW(gg_ttg, 5, 3, 16, 256, {0, 1, 4}),
    ME_ROW(gg_ttgg, 6, 4, 123, 512, {0, 1, 4, 5}), ME_ROW(gg_ttggg, 7, 5, 1240, 1536, {0, 1, 4, 5, 6}),
    // g ubar -> tau+ tau- + (n-1) g + ubar (PAPER.md:110-122 is n = 3): 0 g, 1 ubar, 2 tau+, 3 tau-,
    // 4.. g, last ubar
    { "gux_taptamux", 5, 1, 4, 96, {0}, 0,
      { me_launch_gux_taptamux_p0, me_launch_gux_taptamux_p1, me_launch_gux_taptamux_p2 }, nullptr, nullptr, nullptr, kChanKeys_gux_taptamux },
    { "gux_taptamgux", 6, 2, 16, 96, {0, 4}, 0,
      { me_launch_gux_taptamgux_p0, me_launch_gux_taptamgux_p1, me_launch_gux_taptamgux_p2 }, nullptr, nullptr, nullptr, kChanKeys_gux_taptamgux },
    { "gux_taptamggux", 7, 3, 100, 192, {0, 4, 5}, 0,
      { me_launch_gux_taptamggux_p0, me_launch_gux_taptamggux_p1, me_launch_gux_taptamggux_p2 }, nullptr, nullptr, nullptr, kChanKeys_gux_taptamggux },
};

thread_local std::string g_create_error;

}  // namespace

struct me_handle {
  const ProcDesc* proc;
  int precision, device;
  int npar, ncomb, ncol, denom;
  me::DevParams par;
  bool have_good;
  me::GoodList good;
  // scratch
  double* d_cum;
  size_t cum_bytes;
  unsigned long long* d_frac;
  // lane-group pipeline (gg_ttgg, gg_ttggg): per-event data and jamps between its kernels, one chunk of events
  void* d_scratch;
  size_t scratch_bytes;
  void* d_mc;         // multichannel: per-event data of the diagram kernel (grows on first use)
  size_t mc_bytes;
  me::PipeCtx pipe;   // internal streams / events of the pipeline (valid iff d_scratch)
  bool have_pipe;
  // staging for me_compute_host
  void* d_stage;
  size_t stage_bytes;
  cudaStream_t own_stream, s_in, s_out;   // me_compute_host: compute, copy-in and copy-out streams
  cudaEvent_t ev_in[2], ev_comp[2], ev_out[2];
  me::LaunchInfo last;
  mutable std::string err;
};

namespace {

int fail(const me_handle* h, int code, const std::string& msg) {
  if (h) h->err = msg; else g_create_error = msg;
  return code;
}
int cuda_fail(const me_handle* h, cudaError_t e, const char* where) {
  return fail(h, ME_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
int factorial(int n) { int r = 1; for (int k = 2; k <= n; k++) r *= k; return r; }

// permutations of the gluon particle indices in lexicographic order (reading R8)
void flows_of(const ProcDesc* p, int8_t* out) {
  int gl[8], n = p->ngl;
  for (int k = 0; k < n; k++) gl[k] = p->gluons[k];
  int idx[8];
  for (int k = 0; k < n; k++) idx[k] = k;
  int row = 0;
  while (true) {
    for (int k = 0; k < n; k++) out[row * n + k] = (int8_t)gl[idx[k]];
    row++;
    int i = n - 2;
    while (i >= 0 && idx[i] > idx[i + 1]) i--;
    if (i < 0) break;
    int j = n - 1;
    while (idx[j] < idx[i]) j--;
    int t = idx[i]; idx[i] = idx[j]; idx[j] = t;
    for (int a = i + 1, b = n - 1; a < b; a++, b--) { t = idx[a]; idx[a] = idx[b]; idx[b] = t; }
  }
}

int ensure(me_handle* h, void** p, size_t* have, size_t want) {
  if (*have >= want) return 0;
  if (*p) cudaFree(*p);
  *p = nullptr; *have = 0;
  cudaError_t e = cudaMalloc(p, want);
  if (e != cudaSuccess) return fail(h, ME_ERR_NOMEM, std::string("cudaMalloc: ") + cudaGetErrorString(e));
  *have = want;
  return 0;
}

bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) != 0; }

// Makes the handle's device current for the duration of a call and restores the caller's device on every exit path
struct DeviceGuard {
  int prev;
  cudaError_t err;
  explicit DeviceGuard(int device) : prev(-1), err(cudaSuccess) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
  }
  ~DeviceGuard() {
    int now = -1;
    if (prev >= 0 && cudaGetDevice(&now) == cudaSuccess && now != prev) cudaSetDevice(prev);
  }
};

// Cap of the pipeline scratch of a handle: 2 GiB for gg_ttgg, 8 GiB for gg_ttggg (only batches that want it get there,
// see reserve_scratch), or ME_B200_SCRATCH_MB.  Measured on B200 (round 3, caps 1 / 2 / 4 / 8 GiB): gg_ttggg fp64, 262144
// events per call: 239.4 / 237.7 / 236.8 / 236.3 ms (larger chunks, fewer chunk tails); gg_ttgg fp64, 2^20 events: 47.34 /
// 46.91 / 47.48 / 47.54 ms (beyond 2 GiB the chunks' jamps stop fitting the L2 as well).
size_t scratch_target(int ngluon) {
  const char* s = getenv("ME_B200_SCRATCH_MB");
  long mb = s ? atol(s) : 0;
  if (mb < 16) mb = (ngluon >= 5) ? 8192 : 2048;
  return (size_t)mb << 20;
}

// running helicity sums of the one-event-per-thread kernel [ngood][slots]: sized for the full persistent grid once the
// good-helicity list is known (me_filter_helicities / me_set_good_helicities), so that me_compute never allocates
int size_cum(me_handle* h) {
  me::LaunchArgs a;
  memset(&a, 0, sizeof(a));
  a.nevt = 1ll << 40;  // geometry of the largest grid
  a.good = h->good;
  me::LaunchInfo info;
  memset(&info, 0, sizeof(info));
  int ce = h->proc->fn[h->precision](a, me::MODE_SELECT, nullptr, &info, 1);
  if (ce) return cuda_fail(h, (cudaError_t)ce, "selection scratch geometry");
  if (info.cum_slots <= 0) return 0;
  void* p = h->d_cum;
  int rc = ensure(h, &p, &h->cum_bytes, sizeof(double) * (size_t)h->good.n * (size_t)info.cum_slots);
  h->d_cum = (double*)p;
  return rc;
}

// Pipeline scratch of the lane-group processes for a call of nevt events in `mode`: grows (never shrinks) up to the cap of
// scratch_target(ngluon).  A call whose preferred chunks fit what the handle already owns does not allocate.
int reserve_scratch(me_handle* h, int64_t nevt, int mode) {
  if (!h->have_pipe || nevt <= 0) return 0;
  me::LaunchArgs a;
  memset(&a, 0, sizeof(a));
  a.nevt = nevt;
  a.good = h->good;
  a.good.mask[0] = a.good.mask[1] = h->good.n ? 0ull : ~0ull;   // no list yet (me_reserve before the filter): all rows
  for (int i = 0; i < a.good.n; i++) a.good.mask[a.good.h[i] >> 6] |= 1ull << (a.good.h[i] & 63);
  me::LaunchInfo info;
  memset(&info, 0, sizeof(info));
  int ce = h->proc->fn[mode == me::MODE_FILTER ? 0 : h->precision](a, mode, nullptr, &info, 1);
  if (ce) return cuda_fail(h, (cudaError_t)ce, "pipeline scratch geometry");
  const size_t cap = scratch_target(h->proc->ngl);
  size_t want = (size_t)info.scratch_wanted;
  if (want > cap) want = cap;
  if (want <= h->scratch_bytes) return 0;
  if (want < 2 * h->scratch_bytes) want = (2 * h->scratch_bytes < cap) ? 2 * h->scratch_bytes : cap;   // few growth steps
  return ensure(h, &h->d_scratch, &h->scratch_bytes, want);   // cudaFree waits for the work that still uses the old one
}

}  // namespace

extern "C" {

int me_reserve(me_handle* h, int64_t max_events_per_call) {
  if (!h) return ME_ERR_ARG;
  if (max_events_per_call < 0) return fail(h, ME_ERR_ARG, "me_reserve: negative event count");
  DeviceGuard guard(h->device);
  if (guard.err != cudaSuccess) return cuda_fail(h, guard.err, "me_reserve");
  int rc = reserve_scratch(h, max_events_per_call < 16384 ? max_events_per_call : 16384, me::MODE_FILTER);
  if (!rc) rc = reserve_scratch(h, max_events_per_call, me::MODE_SELECT);
  return rc;
}

int me_create(me_handle** out, const char* process, int precision, const me_params* params, int device) {
  if (!out || !process) return fail(nullptr, ME_ERR_ARG, "me_create: null argument");
  *out = nullptr;
  if (precision < 0 || precision > 2) return fail(nullptr, ME_ERR_ARG, "me_create: precision must be 0, 1 or 2");
  const ProcDesc* pd = nullptr;
  for (const ProcDesc& p : kProcs)
    if (!strcmp(p.name, process)) pd = &p;
  if (!pd) return fail(nullptr, ME_ERR_PROCESS, std::string("me_create: unknown process '") + process + "'");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "me_create: cudaGetDeviceCount (no CUDA device; this library has no CPU path)");
  if (device < 0 || device >= ndev) return fail(nullptr, ME_ERR_ARG, "me_create: bad device ordinal");
  me_handle* h = new (std::nothrow) me_handle();
  if (!h) return fail(nullptr, ME_ERR_NOMEM, "me_create: out of host memory");
  h->proc = pd; h->precision = precision; h->device = device;
  h->npar = pd->npar; h->ncomb = 1 << pd->npar; h->ncol = pd->ngl ? factorial(pd->ngl) : 1;
  h->denom = pd->denom;
  me_params P = {173.0, 1.4915, 91.188, 2.441, 132.507, 1.16639e-5};
  if (params) P = *params;
  h->par.mt = P.mt; h->par.wt = P.wt; h->par.mz = P.mz; h->par.wz = P.wz;
  {  // (alpha, G_F, M_Z) scheme, reading R5
    const double pi = 3.14159265358979323846, alpha = 1.0 / P.aewm1, mz2 = P.mz * P.mz;
    const double mw2 = 0.5 * mz2 + std::sqrt(0.25 * mz2 * mz2 - pi * alpha * mz2 / (std::sqrt(2.0) * P.gf));
    const double sw2 = 1.0 - mw2 / mz2, sc = std::sqrt(sw2 * (1.0 - sw2)), ee = std::sqrt(4.0 * pi * alpha);
    h->par.ee2 = ee * ee; h->par.gl = ee / sc * (sw2 - 0.5); h->par.gr = ee / sc * sw2;
    h->par.glu = ee / sc * (0.5 - (2.0 / 3.0) * sw2); h->par.gru = ee / sc * (-(2.0 / 3.0) * sw2);
  }
  h->have_good = false; h->good.n = 0;
  h->d_cum = nullptr; h->cum_bytes = 0; h->d_frac = nullptr; h->d_stage = nullptr; h->stage_bytes = 0;
  h->d_scratch = nullptr; h->scratch_bytes = 0; h->have_pipe = false; h->d_mc = nullptr; h->mc_bytes = 0;
  memset(&h->pipe, 0, sizeof(h->pipe));
  h->own_stream = nullptr; h->s_in = nullptr; h->s_out = nullptr;
  for (int i = 0; i < 2; i++) { h->ev_in[i] = nullptr; h->ev_comp[i] = nullptr; h->ev_out[i] = nullptr; }
  memset(&h->last, 0, sizeof(h->last));
  DeviceGuard guard(device);
  if ((e = guard.err) != cudaSuccess || (e = cudaMalloc(&h->d_frac, 128 * sizeof(unsigned long long))) != cudaSuccess) {
    int rc = cuda_fail(nullptr, e, "me_create");
    delete h;
    return rc;
  }
  {  // lane-group pipeline: one chunk of scratch, allocated here and never again
    me::LaunchArgs a;
    memset(&a, 0, sizeof(a));
    me::LaunchInfo i0, i1;
    memset(&i0, 0, sizeof(i0)); memset(&i1, 0, sizeof(i1));
    int ce = pd->fn[0](a, me::MODE_FILTER, nullptr, &i0, 1);
    if (!ce) ce = pd->fn[precision](a, me::MODE_SELECT, nullptr, &i1, 1);
    if (ce) {
      int rc = cuda_fail(nullptr, (cudaError_t)ce, "me_create: launch geometry");
      cudaFree(h->d_frac);
      delete h;
      return rc;
    }
    if (i0.scratch_per_event > 0 || i1.scratch_per_event > 0) {
      // the scratch itself is sized by the batches that arrive (reserve_scratch below) or by me_reserve
      // internal streams: two for the setup + amplitude kernels of alternating chunks, a high-priority one for the
      // colour kernels; events carry the dependencies (nothing is synchronised on the host)
      int lo = 0, hi = 0;
      e = cudaDeviceGetStreamPriorityRange(&lo, &hi);
      me::PipeCtx& px = h->pipe;
      if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&px.sa, cudaStreamNonBlocking, lo);
      if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&px.sb, cudaStreamNonBlocking, lo);
      if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&px.s2, cudaStreamNonBlocking, hi);
      cudaEvent_t* evs[7] = {&px.fork, &px.k1[0], &px.k1[1], &px.k2[0], &px.k2[1], &px.k2[2], &px.k2[3]};
      for (int i = 0; i < 7 && e == cudaSuccess; i++) e = cudaEventCreateWithFlags(evs[i], cudaEventDisableTiming);
      if (e != cudaSuccess) {
        int rc = cuda_fail(nullptr, e, "me_create: pipeline streams");
        for (cudaStream_t s : {px.sa, px.sb, px.s2}) if (s) cudaStreamDestroy(s);   // px was zeroed: non-null = created
        for (int i = 0; i < 7; i++) if (*evs[i]) cudaEventDestroy(*evs[i]);
        cudaFree(h->d_frac);
        delete h;
        return rc;
      }
      h->have_pipe = true;
    }
  }
  *out = h;
  return ME_OK;
}

int me_destroy(me_handle* h) {
  if (!h) return ME_ERR_ARG;
  DeviceGuard guard(h->device);
  if (h->have_pipe) {
    cudaStreamDestroy(h->pipe.sa); cudaStreamDestroy(h->pipe.sb); cudaStreamDestroy(h->pipe.s2);
    cudaEventDestroy(h->pipe.fork);
    for (int i = 0; i < 2; i++) cudaEventDestroy(h->pipe.k1[i]);
    for (int i = 0; i < 4; i++) cudaEventDestroy(h->pipe.k2[i]);
  }
  if (h->d_mc) cudaFree(h->d_mc);
  if (h->d_scratch) cudaFree(h->d_scratch);
  if (h->d_cum) cudaFree(h->d_cum);
  if (h->d_frac) cudaFree(h->d_frac);
  if (h->d_stage) cudaFree(h->d_stage);
  if (h->own_stream) {
    cudaStreamDestroy(h->own_stream);
    if (h->s_in) cudaStreamDestroy(h->s_in);
    if (h->s_out) cudaStreamDestroy(h->s_out);
    for (int i = 0; i < 2; i++) {
      if (h->ev_in[i]) cudaEventDestroy(h->ev_in[i]);
      if (h->ev_comp[i]) cudaEventDestroy(h->ev_comp[i]);
      if (h->ev_out[i]) cudaEventDestroy(h->ev_out[i]);
    }
  }
  delete h;
  return ME_OK;
}

const char* me_last_error(const me_handle* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int me_info(const me_handle* h, int* npar, int* ncomb, int* ncol, int* ndiag, int* denom) {
  if (!h) return ME_ERR_ARG;
  if (npar) *npar = h->npar;
  if (ncomb) *ncomb = h->ncomb;
  if (ncol) *ncol = h->ncol;
  if (ndiag) *ndiag = h->proc->ndiag;
  if (denom) *denom = h->denom;
  return ME_OK;
}

int me_helicity_table(const me_handle* h, int8_t* out) {
  if (!h || !out) return fail(h, ME_ERR_ARG, "me_helicity_table: null argument");
  for (int r = 0; r < h->ncomb; r++)
    for (int k = 0; k < h->npar; k++) out[r * h->npar + k] = ((r >> (h->npar - 1 - k)) & 1) ? 1 : -1;
  return ME_OK;
}

int me_color_table(const me_handle* h, int8_t* out) {
  if (!h) return ME_ERR_ARG;
  if (h->proc->ngl == 0) return ME_OK;
  if (!out) return fail(h, ME_ERR_ARG, "me_color_table: null argument");
  flows_of(h->proc, out);
  return ME_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// colour matrix, helicity filter, compute
// ------------------------------------------------------------------------------------------------

namespace {

void cmat_of(const me_handle* h, const int** num, int* den) {
  const char* n = h->proc->name;
  if (!strcmp(n, "ee_mumu")) { *num = kCmat_ee_mumu; *den = kCden_ee_mumu; }
  else if (!strcmp(n, "gg_tt")) { *num = kCmat_gg_tt; *den = kCden_gg_tt; }
  else if (!strcmp(n, "gg_ttg")) { *num = kCmat_gg_ttg; *den = kCden_gg_ttg; }
  else if (!strcmp(n, "gg_ttgg")) { *num = kCmat_gg_ttgg; *den = kCden_gg_ttgg; }
  else if (!strcmp(n, "gux_taptamux")) { *num = kCmat_gux_taptamux; *den = kCden_gux_taptamux; }
  else if (!strcmp(n, "gux_taptamgux")) { *num = kCmat_gux_taptamgux; *den = kCden_gux_taptamgux; }
  else if (!strcmp(n, "gux_taptamggux")) { *num = kCmat_gux_taptamggux; *den = kCden_gux_taptamggux; }
  else { *num = kCmat_gg_ttggg; *den = kCden_gg_ttggg; }
}

int check_inputs(me_handle* h, const double* d_momenta, const double* d_gs, int64_t nevt, const char* who) {
  if (!h) return ME_ERR_ARG;
  if (nevt < 0) return fail(h, ME_ERR_ARG, std::string(who) + ": nevt < 0");
  if (nevt > 0 && (!d_momenta || (h->proc->ngl && !d_gs))) return fail(h, ME_ERR_ARG, std::string(who) + ": null input pointer");
  if (misaligned(d_momenta, 8) || misaligned(d_gs, 8)) return fail(h, ME_ERR_ARG, std::string(who) + ": misaligned input pointer");
  return ME_OK;
}

}  // namespace

extern "C" {

int me_color_matrix(const me_handle* h, double* out) {
  if (!h || !out) return fail(h, ME_ERR_ARG, "me_color_matrix: null argument");
  const int* num; int den;
  cmat_of(h, &num, &den);
  for (int i = 0; i < h->ncol * h->ncol; i++) out[i] = double(num[i]) / double(den);
  return ME_OK;
}

int me_filter_helicities(me_handle* h, const double* d_momenta, const double* d_gs, int64_t nevt, void* stream) {
  int rc = check_inputs(h, d_momenta, d_gs, nevt, "me_filter_helicities");
  if (rc) return rc;
  if (nevt == 0) return fail(h, ME_ERR_ARG, "me_filter_helicities: needs at least one event");
  DeviceGuard guard(h->device);
  cudaError_t e = guard.err;
  if (e != cudaSuccess) return cuda_fail(h, e, "me_filter_helicities");
  cudaStream_t st = (cudaStream_t)stream;
  if ((e = cudaMemsetAsync(h->d_frac, 0, 128 * sizeof(unsigned long long), st)) != cudaSuccess)
    return cuda_fail(h, e, "me_filter_helicities: memset");
  if ((rc = reserve_scratch(h, nevt < 16384 ? nevt : 16384, me::MODE_FILTER)) != 0) return rc;
  me::LaunchArgs a;
  memset(&a, 0, sizeof(a));
  a.mom = d_momenta; a.gs = d_gs; a.nevt = nevt < 16384 ? nevt : 16384;
  a.fracmax = h->d_frac; a.par = h->par;
  a.scratch = h->d_scratch; a.scratch_bytes = h->scratch_bytes; a.pipe = h->have_pipe ? &h->pipe : nullptr;
  int ce = h->proc->fn[0](a, me::MODE_FILTER, stream, nullptr, 0);  // always the fp64 build (reading R10)
  if (ce) return cuda_fail(h, (cudaError_t)ce, "me_filter_helicities: launch");
  unsigned long long bits[128];
  if ((e = cudaMemcpyAsync(bits, h->d_frac, sizeof(bits), cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
      (e = cudaStreamSynchronize(st)) != cudaSuccess)
    return cuda_fail(h, e, "me_filter_helicities: readback");
  h->good.n = 0;
  for (int r = 0; r < h->ncomb; r++) {
    double f;
    memcpy(&f, &bits[r], sizeof(f));
    if (f > 1e-12) h->good.h[h->good.n++] = (uint8_t)r;
  }
  h->have_good = true;
  if (h->good.n == 0) return fail(h, ME_ERR_NO_HELICITIES, "me_filter_helicities: no helicity passed the filter");
  return size_cum(h);
}

int me_get_good_helicities(const me_handle* h, int* ngood, uint8_t* mask) {
  if (!h) return ME_ERR_ARG;
  if (!h->have_good) return fail(h, ME_ERR_NO_HELICITIES, "me_get_good_helicities: no helicity mask yet");
  if (ngood) *ngood = h->good.n;
  if (mask) {
    memset(mask, 0, h->ncomb);
    for (int i = 0; i < h->good.n; i++) mask[h->good.h[i]] = 1;
  }
  return ME_OK;
}

int me_set_good_helicities(me_handle* h, const uint8_t* mask) {
  if (!h || !mask) return fail(h, ME_ERR_ARG, "me_set_good_helicities: null argument");
  int n = 0;
  for (int r = 0; r < h->ncomb; r++) n += mask[r] ? 1 : 0;
  if (n == 0) return fail(h, ME_ERR_ARG, "me_set_good_helicities: empty mask");
  h->good.n = 0;
  for (int r = 0; r < h->ncomb; r++)
    if (mask[r]) h->good.h[h->good.n++] = (uint8_t)r;
  h->have_good = true;
  DeviceGuard guard(h->device);
  if (guard.err != cudaSuccess) return cuda_fail(h, guard.err, "me_set_good_helicities");
  return size_cum(h);
}

static int compute_core(me_handle* h, const double* d_momenta, const double* d_gs, const double* d_rndhel,
                        const double* d_rndcol, int64_t nevt, double* d_me, int32_t* d_selhel, int32_t* d_selcol,
                        void* stream, const int32_t* d_channel, const unsigned* d_chanflows, int nchan) {
  int rc = check_inputs(h, d_momenta, d_gs, nevt, "me_compute");
  if (rc) return rc;
  if (!h->have_good) return fail(h, ME_ERR_NO_HELICITIES, "me_compute: call me_filter_helicities or me_set_good_helicities first");
  if (nevt > 0 && !d_me) return fail(h, ME_ERR_ARG, "me_compute: null output pointer");
  if (misaligned(d_me, 8) || misaligned(d_rndhel, 8) || misaligned(d_rndcol, 8) || misaligned(d_selhel, 4) || misaligned(d_selcol, 4))
    return fail(h, ME_ERR_ARG, "me_compute: misaligned pointer");
  if ((d_selhel && !d_rndhel) || (d_selcol && !d_rndcol))
    return fail(h, ME_ERR_ARG, "me_compute: a selection output needs its random-number input");
  if (nevt == 0) return ME_OK;
  DeviceGuard guard(h->device);
  if (guard.err != cudaSuccess) return cuda_fail(h, guard.err, "me_compute");
  if ((rc = reserve_scratch(h, nevt, me::MODE_SELECT)) != 0) return rc;   // allocates only for a batch larger than any before
  me::LaunchArgs a;
  memset(&a, 0, sizeof(a));
  a.mom = d_momenta; a.gs = d_gs; a.rndhel = d_rndhel; a.rndcol = d_rndcol; a.nevt = nevt;
  a.me = d_me; a.selhel = d_selhel; a.selcol = d_selcol; a.par = h->par; a.good = h->good;
  a.scratch = h->d_scratch; a.scratch_bytes = h->scratch_bytes; a.pipe = h->have_pipe ? &h->pipe : nullptr;
  a.channel = d_channel; a.chanflows = d_chanflows; a.nchan = nchan;
  a.good.mask[0] = a.good.mask[1] = 0ull;
  for (int i = 0; i < a.good.n; i++) a.good.mask[a.good.h[i] >> 6] |= 1ull << (a.good.h[i] & 63);
  const int mode = (d_selhel || d_selcol) ? me::MODE_SELECT : me::MODE_ME;
  launch_fn fn = h->proc->fn[h->precision];
  me::LaunchInfo info;
  int ce = fn(a, mode, stream, &info, 1);
  if (ce) return cuda_fail(h, (cudaError_t)ce, "me_compute: launch geometry");
  if (mode == me::MODE_SELECT && info.cum_slots > 0) {
    // running helicity sums [ngood][slots], sized by me_filter_helicities / me_set_good_helicities
    if (sizeof(double) * (size_t)h->good.n * (size_t)info.cum_slots > h->cum_bytes)
      return fail(h, ME_ERR_ARG, "me_compute: selection scratch smaller than the grid (internal)");
    a.cum = h->d_cum;
  }
  a.blocks = info.blocks;
  ce = fn(a, mode, stream, nullptr, 0);
  if (ce) return cuda_fail(h, (cudaError_t)ce, "me_compute: launch");
  h->last = info;
  return ME_OK;
}

int me_compute(me_handle* h, const double* d_momenta, const double* d_gs, const double* d_rndhel,
               const double* d_rndcol, int64_t nevt, double* d_me, int32_t* d_selhel, int32_t* d_selcol,
               void* stream) {
  return compute_core(h, d_momenta, d_gs, d_rndhel, d_rndcol, nevt, d_me, d_selhel, d_selcol, stream, nullptr, nullptr, 0);
}

int me_compute_multichannel(me_handle* h, const double* d_momenta, const double* d_gs, const double* d_rndhel,
                            const double* d_rndcol, const int32_t* d_channel, int64_t nevt, double* d_me,
                            int32_t* d_selhel, int32_t* d_selcol, double* d_num, double* d_den, void* stream) {
  if (!h) return ME_ERR_ARG;
  if (!h->proc->diag) return fail(h, ME_ERR_PROCESS, "me_compute_multichannel: no channels for this process");
  if (nevt > 0 && (!d_channel || !d_num || !d_den)) return fail(h, ME_ERR_ARG, "me_compute_multichannel: null channel / num / den pointer");
  if (misaligned(d_channel, 4) || misaligned(d_num, 8) || misaligned(d_den, 8)) return fail(h, ME_ERR_ARG, "me_compute_multichannel: misaligned pointer");
  DeviceGuard guard(h->device);
  if (guard.err != cudaSuccess) return cuda_fail(h, guard.err, "me_compute_multichannel");
  const unsigned* cfl = nullptr;
  int nchan = 0;
  int ce = h->proc->chanflows(&cfl, &nchan);
  if (ce) return cuda_fail(h, (cudaError_t)ce, "me_compute_multichannel: channel table");
  // the matrix element, with the colour selection restricted to the flows of each event's channel
  int rc = compute_core(h, d_momenta, d_gs, d_rndhel, d_rndcol, nevt, d_me, d_selhel, d_selcol, stream, d_channel, cfl, nchan);
  if (rc || nevt == 0) return rc;
  // the single-diagram-enhancement weights: diagram-by-diagram kernel, fp64 whatever the build, in chunks that fit its scratch
  const size_t per = h->proc->diag_scratch();
  int64_t chunk = nevt < 65536 ? nevt : 65536;
  void* p = h->d_mc;
  rc = ensure(h, &p, &h->mc_bytes, per * (size_t)chunk);
  h->d_mc = p;
  if (rc) return rc;
  me::LaunchArgs a;
  memset(&a, 0, sizeof(a));
  a.par = h->par; a.good = h->good;
  for (int64_t e0 = 0; e0 < nevt; e0 += chunk) {
    a.nevt = (nevt - e0 < chunk) ? (nevt - e0) : chunk;
    a.mom = d_momenta + e0 * h->npar * 4; a.gs = d_gs + e0;
    ce = h->proc->diag(a, d_channel + e0, d_num + e0, d_den + e0, h->d_mc, stream);
    if (ce) return cuda_fail(h, (cudaError_t)ce, "me_compute_multichannel: launch");
  }
  return ME_OK;
}

int me_channel_table(const me_handle* h, char* out, int cap) {
  if (!h) return ME_ERR_ARG;
  const int need = (int)strlen(h->proc->chan_keys) + 1;
  if (out && cap >= need) memcpy(out, h->proc->chan_keys, (size_t)need);
  else if (out) return fail(h, ME_ERR_ARG, "me_channel_table: buffer too small");
  return need;
}

int me_compute_host(me_handle* h, const double* momenta, const double* gs, const double* rndhel,
                    const double* rndcol, int64_t nevt, double* me_out, int32_t* selhel, int32_t* selcol) {
  if (!h) return ME_ERR_ARG;
  if (nevt < 0) return fail(h, ME_ERR_ARG, "me_compute_host: nevt < 0");
  if (nevt == 0) return ME_OK;
  if (!momenta || !me_out || (h->proc->ngl && !gs)) return fail(h, ME_ERR_ARG, "me_compute_host: null pointer");
  DeviceGuard guard(h->device);
  cudaError_t e = guard.err;
  if (e != cudaSuccess) return cuda_fail(h, e, "me_compute_host");
  if (!h->own_stream) {
    // three internal streams (copy in, compute, copy out) and the events that chain them, made once
    if ((e = cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking)) != cudaSuccess ||
        (e = cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking)) != cudaSuccess ||
        (e = cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking)) != cudaSuccess)
      return cuda_fail(h, e, "me_compute_host: stream");
    for (int i = 0; i < 2; i++)
      if ((e = cudaEventCreateWithFlags(&h->ev_in[i], cudaEventDisableTiming)) != cudaSuccess ||
          (e = cudaEventCreateWithFlags(&h->ev_comp[i], cudaEventDisableTiming)) != cudaSuccess ||
          (e = cudaEventCreateWithFlags(&h->ev_out[i], cudaEventDisableTiming)) != cudaSuccess)
        return cuda_fail(h, e, "me_compute_host: event");
  }
  // Chunks of the batch flow through two staging slots: while chunk k is computed, chunk k + 1 is copied in and the
  // results of chunk k - 1 are copied out (one cudaMemcpyAsync per array and chunk).
  int64_t chunk = (nevt + 7) / 8;
  if (chunk < 16384) chunk = 16384;
  if (chunk > 262144) chunk = 262144;
  if (chunk > nevt) chunk = nevt;
  const size_t c = (size_t)chunk, bm = c * h->npar * 4 * 8, b8 = c * 8, b4 = c * 4;
  // layout of one staging slot: momenta | gs | rndhel | rndcol | me | selhel | selcol
  const size_t slot = ((bm + 4 * b8 + 2 * b4 + 255) / 256) * 256;
  int rc = ensure(h, &h->d_stage, &h->stage_bytes, 2 * slot);
  if (rc) return rc;
  const bool sh = selhel && rndhel, sc = selcol && rndcol;
  // error exit of the chunk loop: earlier chunks may still be copying into the caller's buffers or using the staging slots;
  // nothing may be in flight when the caller gets control back
  auto drain = [h](int code) {
    cudaStreamSynchronize(h->s_in); cudaStreamSynchronize(h->own_stream); cudaStreamSynchronize(h->s_out);
    return code;
  };
  // the first chunk is an eighth of the others: its copy-in is the only one no kernel hides
  const int64_t first = (chunk / 8 > 4096) ? chunk / 8 : chunk;
  int64_t k = 0, n = 0;
  for (int64_t e0 = 0; e0 < nevt; e0 += n, k++) {
    n = (k == 0) ? first : chunk;
    if (n > nevt - e0) n = nevt - e0;
    const int b = (int)(k & 1);
    char* base = (char*)h->d_stage + (size_t)b * slot;
    double* d_mom = (double*)base;
    double* d_gs = (double*)(base + bm);
    double* d_rh = (double*)(base + bm + b8);
    double* d_rc = (double*)(base + bm + 2 * b8);
    double* d_me = (double*)(base + bm + 3 * b8);
    int32_t* d_sh = (int32_t*)(base + bm + 4 * b8);
    int32_t* d_sc = (int32_t*)(base + bm + 4 * b8 + b4);
    const size_t nn = (size_t)n;
    // copy in (the slot's inputs are free once the compute of chunk k - 2 has finished)
    if (k >= 2 && (e = cudaStreamWaitEvent(h->s_in, h->ev_comp[b], 0)) != cudaSuccess) return drain(cuda_fail(h, e, "me_compute_host: wait"));
    if ((e = cudaMemcpyAsync(d_mom, momenta + (size_t)e0 * h->npar * 4, nn * h->npar * 32, cudaMemcpyHostToDevice, h->s_in)) != cudaSuccess) return drain(cuda_fail(h, e, "H2D momenta"));
    if (gs && (e = cudaMemcpyAsync(d_gs, gs + e0, nn * 8, cudaMemcpyHostToDevice, h->s_in)) != cudaSuccess) return drain(cuda_fail(h, e, "H2D gs"));
    if (sh && (e = cudaMemcpyAsync(d_rh, rndhel + e0, nn * 8, cudaMemcpyHostToDevice, h->s_in)) != cudaSuccess) return drain(cuda_fail(h, e, "H2D rndhel"));
    if (sc && (e = cudaMemcpyAsync(d_rc, rndcol + e0, nn * 8, cudaMemcpyHostToDevice, h->s_in)) != cudaSuccess) return drain(cuda_fail(h, e, "H2D rndcol"));
    if ((e = cudaEventRecord(h->ev_in[b], h->s_in)) != cudaSuccess) return drain(cuda_fail(h, e, "me_compute_host: record"));
    // compute (the slot's outputs are free once the copy-out of chunk k - 2 has finished)
    if ((e = cudaStreamWaitEvent(h->own_stream, h->ev_in[b], 0)) != cudaSuccess) return drain(cuda_fail(h, e, "me_compute_host: wait"));
    if (k >= 2 && (e = cudaStreamWaitEvent(h->own_stream, h->ev_out[b], 0)) != cudaSuccess) return drain(cuda_fail(h, e, "me_compute_host: wait"));
    rc = me_compute(h, d_mom, gs ? d_gs : nullptr, sh ? d_rh : nullptr, sc ? d_rc : nullptr, n, d_me,
                    sh ? d_sh : nullptr, sc ? d_sc : nullptr, h->own_stream);
    if (rc) return drain(rc);
    if ((e = cudaEventRecord(h->ev_comp[b], h->own_stream)) != cudaSuccess) return drain(cuda_fail(h, e, "me_compute_host: record"));
    // copy out
    if ((e = cudaStreamWaitEvent(h->s_out, h->ev_comp[b], 0)) != cudaSuccess) return drain(cuda_fail(h, e, "me_compute_host: wait"));
    if ((e = cudaMemcpyAsync(me_out + e0, d_me, nn * 8, cudaMemcpyDeviceToHost, h->s_out)) != cudaSuccess) return drain(cuda_fail(h, e, "D2H me"));
    if (sh && (e = cudaMemcpyAsync(selhel + e0, d_sh, nn * 4, cudaMemcpyDeviceToHost, h->s_out)) != cudaSuccess) return drain(cuda_fail(h, e, "D2H selhel"));
    if (sc && (e = cudaMemcpyAsync(selcol + e0, d_sc, nn * 4, cudaMemcpyDeviceToHost, h->s_out)) != cudaSuccess) return drain(cuda_fail(h, e, "D2H selcol"));
    if ((e = cudaEventRecord(h->ev_out[b], h->s_out)) != cudaSuccess) return drain(cuda_fail(h, e, "me_compute_host: record"));
  }
  if ((e = cudaStreamSynchronize(h->s_out)) != cudaSuccess || (e = cudaStreamSynchronize(h->own_stream)) != cudaSuccess ||
      (e = cudaStreamSynchronize(h->s_in)) != cudaSuccess)
    return cuda_fail(h, e, "me_compute_host: synchronize");
  return ME_OK;
}

int me_generate(me_handle* h, uint64_t seed, int64_t start, int64_t nevt, double sqrts, double alphas,
                double* d_momenta, double* d_gs, double* d_rndhel, double* d_rndcol, double* d_weight, void* stream) {
  if (!h) return ME_ERR_ARG;
  if (nevt < 0 || start < 0) return fail(h, ME_ERR_ARG, "me_generate: negative nevt or start");
  if (!(sqrts > 0.0)) return fail(h, ME_ERR_ARG, "me_generate: sqrts must be positive");
  if (nevt > 0 && !d_momenta) return fail(h, ME_ERR_ARG, "me_generate: null momenta pointer");
  if (misaligned(d_momenta, 8) || misaligned(d_gs, 8) || misaligned(d_rndhel, 8) || misaligned(d_rndcol, 8) || misaligned(d_weight, 8))
    return fail(h, ME_ERR_ARG, "me_generate: misaligned pointer");
  const int nfin = h->npar - 2;
  me::RamboArgs a;
  memset(&a, 0, sizeof(a));
  a.mom = d_momenta; a.gs = d_gs; a.rndhel = d_rndhel; a.rndcol = d_rndcol; a.weight = d_weight;
  a.nevt = nevt; a.start = start; a.sqrts = sqrts; a.alphas = alphas;
  double msum = 0.0;
  for (int i = 0; i < nfin; i++) { a.mass[i] = (i < h->proc->nmassive) ? h->par.mt : 0.0; msum += a.mass[i]; }
  if (!(msum < sqrts)) return fail(h, ME_ERR_ARG, "me_generate: sqrts below the mass threshold");
  DeviceGuard guard(h->device);
  if (guard.err != cudaSuccess) return cuda_fail(h, guard.err, "me_generate");
  int ce = me::launch_rambo(a, nfin, (unsigned long long)seed, stream);
  if (ce) return cuda_fail(h, (cudaError_t)ce, "me_generate: launch");
  return ME_OK;
}

int me_launch_info(const me_handle* h, int* threads, int* blocks, int* regs, int* local_bytes) {
  if (!h) return ME_ERR_ARG;
  if (threads) *threads = h->last.threads;
  if (blocks) *blocks = h->last.blocks;
  if (regs) *regs = h->last.regs;
  if (local_bytes) *local_bytes = h->last.local_bytes;
  return ME_OK;
}

int me_launch_stats(const me_handle* h, int* launches, int64_t* chunk_events, int64_t* scratch_bytes) {
  if (!h) return ME_ERR_ARG;
  if (launches) *launches = h->last.launches;
  if (chunk_events) *chunk_events = h->last.chunk;
  if (scratch_bytes) *scratch_bytes = (int64_t)h->scratch_bytes;
  return ME_OK;
}

}  // extern "C"
