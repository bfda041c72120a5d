// me_noalloc.cu -- me_compute_noalloc of include/me_b200.h: gg -> t tbar g in fp64 with helicity and colour selection,
// for callers that must not allocate device memory.
//
// Who that is: code running inside a host application that has already handed the whole GPU to its own memory pool (an
// event generator or an ML framework that reserves its arena up front, or a process held to a fixed memory budget under
// MPS), where a cudaMalloc from a library either fails or eats into a budget the library knows nothing about; and code in
// a latency-critical loop next to other streams, where cudaMalloc / cudaFree may stall the whole device.  The
// normal path cannot serve them: me_create and me_set_good_helicities allocate (handle tables, the running helicity
// sums of the selection).  This entry point needs no handle and calls no cudaMalloc, cudaFree or allocating library
// routine, on the first call or later.
//
// The kernel is the one-event-per-thread kernel of me_kernels.cuh in its selection mode, which needs scratch: the
// running sums over the good helicities, one double per (good helicity, event), written in the helicity loop and read
// back when the helicity is drawn.  Here that scratch is the file-scope device array g_cum below, sized for
// ME_NOALLOC_MAX_EVENTS events and all 32 helicity combinations: 4 MiB, which every GPU that loads libme_b200.so
// holds until the process exits, whether the entry point is used or not.
//
// g_cum in HOST code is only a stand-in the runtime knows the array by, not a device address; handing it to a kernel
// would make the kernel fault (or, where the GPU can reach host memory, scribble over host memory).  The address the
// kernel needs comes from cudaGetSymbolAddress, asked once per device with that device current (scratch_of below).
//
// What stays outside the library's hands: this kernel spills registers (1.7 KB of local memory per thread, as in
// me_compute), and the CUDA driver itself sets that spill space up when a kernel that needs it is first launched.
//
// Compiled with the flags of the gg_ttg fp64 unit of build.py (same generated source, same arithmetic as me_compute).
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "../../include/me_b200.h"
#include "me_kernels.cuh"
#include "gen/proc_gg_ttg.cuh"

namespace {

typedef Proc_gg_ttg Proc;
constexpr int NT = 128;                                      // threads per block = events per tile
constexpr long long MAXEVT = ME_NOALLOC_MAX_EVENTS;
static_assert(MAXEVT % NT == 0, "the slot count of a full grid must equal the event limit");

// [good helicity][slot], slot = event of the call (one tile per block, so a slot serves one event).  Shared by every
// call on the device; nothing in it has to start at zero (each thread writes its column before it reads it).
static __device__ __align__(256) double g_cum[Proc::ncomb * MAXEVT];

// colour-matrix numerators (integers) of this unit
__constant__ double c_cmat_noalloc[Proc::ncol * Proc::ncol] = ME_CMAT_GG_TTG;
struct CMat {
  __device__ __forceinline__ static double at(int i) { return c_cmat_noalloc[i]; }
};

constexpr int MAXDEV = 64;
std::mutex g_mu;
double* g_cum_addr[MAXDEV];   // device address of g_cum on each ordinal, nullptr until the first call there

int fail(char* errbuf, int errcap, int code, const char* msg, const char* detail = nullptr) {
  if (errbuf && errcap > 0) snprintf(errbuf, (size_t)errcap, "me_compute_noalloc: %s%s%s", msg, detail ? ": " : "", detail ? detail : "");
  return code;
}

// Set-up, once per device: the device address of g_cum on the CURRENT device.
cudaError_t scratch_of(int dev, double** out) {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_cum_addr[dev]) {
    double* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_cum);
    if (e != cudaSuccess) return e;
    g_cum_addr[dev] = p;
  }
  *out = g_cum_addr[dev];
  return cudaSuccess;
}

bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) != 0; }

}  // namespace

extern "C" int me_compute_noalloc(const me_params* params, const uint8_t* good_mask, const double* d_momenta,
                                  const double* d_gs, const double* d_rndhel, const double* d_rndcol, int64_t nevt,
                                  double* d_me, int32_t* d_selhel, int32_t* d_selcol, void* stream, char* errbuf,
                                  int errcap) {
  if (errbuf && errcap > 0) errbuf[0] = 0;
  if (nevt < 0) return fail(errbuf, errcap, ME_ERR_ARG, "nevt < 0");
  if (nevt > MAXEVT) {
    char d[160];
    snprintf(d, sizeof(d), "%lld events asked, the static scratch holds %lld (ME_NOALLOC_MAX_EVENTS); split the batch or use me_compute",
             (long long)nevt, MAXEVT);
    return fail(errbuf, errcap, ME_ERR_ARG, "batch too large", d);
  }
  if (nevt > 0 && (!d_momenta || !d_gs || !d_me)) return fail(errbuf, errcap, ME_ERR_ARG, "null momenta / gs / me pointer");
  if (misaligned(d_momenta, 8) || misaligned(d_gs, 8) || misaligned(d_me, 8) || misaligned(d_rndhel, 8) ||
      misaligned(d_rndcol, 8) || misaligned(d_selhel, 4) || misaligned(d_selcol, 4))
    return fail(errbuf, errcap, ME_ERR_ARG, "misaligned pointer");
  if ((d_selhel && !d_rndhel) || (d_selcol && !d_rndcol))
    return fail(errbuf, errcap, ME_ERR_ARG, "a selection output needs its random-number input");
  me::LaunchArgs a;
  memset(&a, 0, sizeof(a));
  for (int r = 0; r < Proc::ncomb; r++)
    if (!good_mask || good_mask[r]) a.good.h[a.good.n++] = (uint8_t)r;
  if (a.good.n == 0) return fail(errbuf, errcap, ME_ERR_NO_HELICITIES, "empty good-helicity mask");
  for (int i = 0; i < a.good.n; i++) a.good.mask[a.good.h[i] >> 6] |= 1ull << (a.good.h[i] & 63);
  if (nevt == 0) return ME_OK;
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(errbuf, errcap, ME_ERR_CUDA, "cudaGetDevice (no CUDA device; this library has no CPU path)", cudaGetErrorString(e));
  if (dev < 0 || dev >= MAXDEV) return fail(errbuf, errcap, ME_ERR_ARG, "device ordinal beyond 63");
  double* cum = nullptr;
  if ((e = scratch_of(dev, &cum)) != cudaSuccess) return fail(errbuf, errcap, ME_ERR_CUDA, "cudaGetSymbolAddress", cudaGetErrorString(e));
  me_params P = {173.0, 1.4915, 91.188, 2.441, 132.507, 1.16639e-5};
  if (params) P = *params;
  a.par.mt = P.mt; a.par.wt = P.wt; a.par.mz = P.mz; a.par.wz = P.wz;   // a pure QCD process: nothing else is read
  a.mom = d_momenta; a.gs = d_gs; a.rndhel = d_rndhel; a.rndcol = d_rndcol; a.nevt = nevt;
  a.me = d_me; a.selhel = d_selhel; a.selcol = d_selcol;
  a.cum = cum;
  // one tile of NT events per block: blocks * NT slots <= ME_NOALLOC_MAX_EVENTS, the extent of g_cum per helicity
  const unsigned blocks = (unsigned)((nevt + NT - 1) / NT);
  me::event_kernel<Proc, double, double, CMat, me::MODE_SELECT, NT, 1><<<blocks, NT, 0, (cudaStream_t)stream>>>(a);
  if ((e = cudaGetLastError()) != cudaSuccess) return fail(errbuf, errcap, ME_ERR_CUDA, "launch", cudaGetErrorString(e));
  return ME_OK;
}
