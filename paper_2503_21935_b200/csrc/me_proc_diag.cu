// me_proc_diag.cu -- one translation unit per gg process: the multichannel (single-diagram-enhancement) kernel of
// me_diag.cuh with the tables of gen/diag_<name>.cuh.   -DME_PROC=<name>
// exports  me_launch_diag_<name>  and  me_chanflows_<name>  (C++ linkage, called from me_api.cu).
#include "me_diag.cuh"

#define ME_CAT_(a, b) a##b
#define ME_CAT(a, b) ME_CAT_(a, b)
#define ME_STR_(x) #x
#define ME_STR(x) ME_STR_(x)

#include ME_STR(ME_CAT(gen/diag_, ME_PROC).cuh)

typedef ME_CAT(Diag_, ME_PROC) Diag;

// scratch bytes per event (the GrpEvent made by setup_kernel); the caller provides scratch for the events of one call
size_t ME_CAT(me_diag_scratch_, ME_PROC)() { return sizeof(me::GrpEvent<double, Diag::n>); }

// device table [nchan][4] of allowed colour flows (bit c), for the channel-restricted colour selection
int ME_CAT(me_chanflows_, ME_PROC)(const unsigned** out, int* nchan) {
  void* sym = nullptr;
  cudaError_t err = cudaGetSymbolAddress(&sym, ME_CAT(kDiagFlows_, ME_PROC));
  *out = (const unsigned*)sym;
  *nchan = Diag::nchan;
  return (int)err;
}

// a: mom, gs, nevt, good list, par; scratch >= nevt * me_diag_scratch bytes
int ME_CAT(me_launch_diag_, ME_PROC)(const me::LaunchArgs& a, const int* d_channel, double* d_num, double* d_den, void* scratch,
                                     void* stream) {
  typedef me::GrpEvent<double, Diag::n> EV;
  typedef me::DiagGeom<Diag> DG;
  cudaStream_t st = (cudaStream_t)stream;
  if (a.nevt == 0) return 0;
  constexpr int PT = ((1 << Diag::n) + Diag::n + 6 <= 32) ? 32 : 64;
  me::setup_kernel<double, Diag::n><<<(unsigned)((a.nevt * PT + 127) / 128), 128, 0, st>>>(a, (EV*)scratch);
  auto k = me::diag_kernel<Diag>;
  // shared-memory limit and persistent-grid size of the kernel, set once per device (not per call)
  static int grid_cached[64];   // SMs x resident blocks per SM on each device ordinal, 0 = not set up yet
  int dev = 0;
  cudaError_t err = cudaGetDevice(&dev);
  if (err != cudaSuccess) return (int)err;
  if (dev < 0 || dev >= 64) return (int)cudaErrorInvalidDevice;
  if (grid_cached[dev] == 0) {
    int sms = 0, per_sm = 1;
    err = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, DG::SMEM);
    if (err == cudaSuccess) err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (err == cudaSuccess) err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, DG::NT, DG::SMEM);
    if (err != cudaSuccess) return (int)err;
    grid_cached[dev] = sms * (per_sm < 1 ? 1 : per_sm);
  }
  long long blocks = grid_cached[dev];
  if (blocks > a.nevt) blocks = a.nevt;
  me::DiagArgs p;
  p.a = a; p.ev = scratch; p.channel = d_channel; p.num = d_num; p.den = d_den;
  k<<<(unsigned)blocks, DG::NT, DG::SMEM, st>>>(p);
  return (int)cudaGetLastError();
}
