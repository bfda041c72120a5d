// me_proc.cu -- one translation unit per (process, precision): compiled with
//   -DME_PROC=<name> -DME_PROC_UP=<NAME> -DME_PREC=<0|1|2> [-DME_NT=<threads>] [-DME_MINB=<min blocks/SM>]
// and exports  me_launch_<name>_p<prec>  (C++ linkage, called from me_api.cu).
// ME_PREC: 0 = fp64 (amplitudes and colour sum in double), 1 = fp32 (both float), 2 = mixed (amplitudes
// double, colour quadratic form float: PAPER.md:108).
#include "me_kernels.cuh"

#define ME_CAT_(a, b) a##b
#define ME_CAT(a, b) ME_CAT_(a, b)
#define ME_STR_(x) #x
#define ME_STR(x) ME_STR_(x)

#if defined(ME_IS_EE_MUMU)
#include "proc_ee_mumu.cuh"
#else
#include ME_STR(ME_CAT(gen/proc_, ME_PROC).cuh)
#endif

#ifndef ME_NT
#define ME_NT 128
#endif
#ifndef ME_MINB
#define ME_MINB 1
#endif
#ifdef ME_MINB_OVERRIDE   // experiments (ME_B200_NVCC_FLAGS): register cap through the minimum number of resident blocks
#undef ME_MINB
#define ME_MINB ME_MINB_OVERRIDE
#endif
#ifdef ME_NT_OVERRIDE
#undef ME_NT
#define ME_NT ME_NT_OVERRIDE
#endif

#if ME_PREC == 0
typedef double T_amp;
typedef double T_col;
#elif ME_PREC == 1
typedef float T_amp;
typedef float T_col;
#else
typedef double T_amp;
typedef float T_col;
#endif

typedef ME_CAT(Proc_, ME_PROC) Proc;

// colour-matrix numerators: integers, exactly representable in fp32 (<= 4096), as T_col
__constant__ T_col c_cmat[Proc::ncol * Proc::ncol] = ME_CAT(ME_CMAT_, ME_PROC_UP);
struct CMat {
  __device__ __forceinline__ static T_col at(int i) { return c_cmat[i]; }
};

template <int MODE, typename TA, typename TCo>
static int launch_mode(const me::LaunchArgs& a, cudaStream_t st, me::LaunchInfo* info, bool dry) {
  auto kern = me::event_kernel<Proc, TA, TCo, CMat, MODE, ME_NT, ME_MINB>;
  // size of the persistent grid, asked once per device (not per call)
  static int grid_cached[64];   // SMs x resident blocks per SM on each device ordinal, 0 = not asked yet
  int dev = 0;
  cudaError_t err = cudaGetDevice(&dev);
  if (err != cudaSuccess) return (int)err;
  if (dev < 0 || dev >= 64) return (int)cudaErrorInvalidDevice;
  if (grid_cached[dev] == 0) {
    int sms = 0, per_sm = 0;
    err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (err == cudaSuccess) err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, ME_NT, 0);
    if (err != cudaSuccess) return (int)err;
    grid_cached[dev] = sms * (per_sm < 1 ? 1 : per_sm);
  }
  long long ntiles = (a.nevt + ME_NT - 1) / ME_NT;
  long long blocks = grid_cached[dev];
  if (a.blocks > 0) blocks = a.blocks;
  if (blocks > ntiles) blocks = ntiles;
  if (blocks < 1) blocks = 1;
  if (info) {
    cudaFuncAttributes fa;
    err = cudaFuncGetAttributes(&fa, kern);
    if (err != cudaSuccess) return (int)err;
    info->threads = ME_NT;
    info->blocks = (int)blocks;
    info->regs = fa.numRegs;
    info->local_bytes = (int)fa.localSizeBytes;
    info->cum_slots = blocks * ME_NT;
    info->scratch_per_event = 0;
    info->chunk = 0;
    info->scratch_wanted = 0;
    info->launches = (a.nevt > 0) ? 1 : 0;
  }
  if (dry || a.nevt == 0) return 0;
  kern<<<(unsigned)blocks, ME_NT, 0, st>>>(a);
  return (int)cudaGetLastError();
}

// mode: me::MODE_*; dry = only report the launch geometry (blocks x threads) in *info.
// The filter always runs in fp64 (reading R10).  Returns a cudaError_t value.
int ME_CAT(ME_CAT(me_launch_, ME_PROC), ME_CAT(_p, ME_PREC))(const me::LaunchArgs& a, int mode, void* stream,
                                                              me::LaunchInfo* info, int dry) {
  cudaStream_t st = (cudaStream_t)stream;
  switch (mode) {
    case me::MODE_ME: return launch_mode<me::MODE_ME, T_amp, T_col>(a, st, info, dry != 0);
    case me::MODE_SELECT: return launch_mode<me::MODE_SELECT, T_amp, T_col>(a, st, info, dry != 0);
#if ME_PREC == 0
    case me::MODE_FILTER: return launch_mode<me::MODE_FILTER, double, double>(a, st, info, dry != 0);
#endif
    default: return (int)cudaErrorInvalidValue;
  }
}
