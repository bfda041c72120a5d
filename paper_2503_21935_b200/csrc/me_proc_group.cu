// me_proc_group.cu -- one translation unit per (process, precision) in the lane-group layout (me_group.cuh):
//   -DME_PROC=<name> -DME_PROC_UP=<NAME> -DME_PREC=<0|1|2> [-DME_MINB=<min blocks/SM>]
// exports  me_launch_<name>_p<prec>  (C++ linkage, called from me_api.cu), same contract as me_proc.cu.
#include "me_group.cuh"

#define ME_CAT_(a, b) a##b
#define ME_CAT(a, b) ME_CAT_(a, b)
#define ME_STR_(x) #x
#define ME_STR(x) ME_STR_(x)

#include ME_STR(ME_CAT(gen/grp_, ME_PROC).cuh)
#include ME_STR(ME_CAT(gen/cmat_, ME_PROC).h)

#ifndef ME_MINB
#define ME_MINB 1
#endif
#ifndef ME_CMAT_GLOBAL
#define ME_CMAT_GLOBAL 0
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

typedef ME_CAT(Grp_, ME_PROC) Grp;

// colour-matrix numerators: integers, exactly representable in fp32 (<= 4096), as T_col
// (constant memory up to 24 flows; the 120 x 120 matrix exceeds the 64 KB bank and is read through L1)
#if ME_CMAT_GLOBAL
__device__ const T_col c_cmat[Grp::ncol * Grp::ncol] = ME_CAT(ME_CMAT_, ME_PROC_UP);
// the same numerators as 16-bit integers (|C| <= 4096): 28.8 KB, copied into shared memory by builds whose
// amplitudes are fp64 (one block per SM anyway); the fp32 build keeps two blocks per SM and reads C through L1
__device__ const short c_cmat16[Grp::ncol * Grp::ncol] = ME_CAT(ME_CMAT_, ME_PROC_UP);
struct CMat {
  static constexpr bool smem16 = (ME_PREC != 1);
  __device__ __forceinline__ static T_col at(int i) { return __ldg(c_cmat + i); }
  __device__ __forceinline__ static const short* table16() { return c_cmat16; }
};
#else
__constant__ T_col c_cmat[Grp::ncol * Grp::ncol] = ME_CAT(ME_CMAT_, ME_PROC_UP);
struct CMat {
  static constexpr bool smem16 = false;
  __device__ __forceinline__ static T_col at(int i) { return c_cmat[i]; }
  __device__ __forceinline__ static const short* table16() { return nullptr; }
};
#endif

template <int MODE, typename TA, typename TCo>
static int launch_mode(const me::LaunchArgs& a, cudaStream_t st, me::LaunchInfo* info, bool dry) {
  typedef me::GrpGeom<Grp, TA> GE;
  auto kern = me::group_kernel<Grp, TA, TCo, CMat, MODE, ME_MINB>;
  const size_t ev_bytes = ((sizeof(me::GrpEvent<TA, TCo, Grp::n>) + 127) / 128) * 128;
  const size_t smem = ev_bytes + (size_t)GE::NPASS * GE::GS * sizeof(TA) + (CMat::smem16 ? (size_t)Grp::ncol * Grp::ncol * 2 + 16 : 0);
  cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (err != cudaSuccess) return (int)err;
  long long blocks = a.nevt;
  if (a.blocks > 0) blocks = a.blocks;
  if (blocks > (1ll << 30)) blocks = 1ll << 30;
  if (blocks < 1) blocks = 1;
  if (info) {
    cudaFuncAttributes fa;
    err = cudaFuncGetAttributes(&fa, kern);
    if (err != cudaSuccess) return (int)err;
    info->threads = GE::NT;
    info->blocks = (int)blocks;
    info->regs = fa.numRegs;
    info->local_bytes = (int)fa.localSizeBytes;
    info->cum_slots = 0;
  }
  if (dry || a.nevt == 0) return 0;
  kern<<<(unsigned)blocks, GE::NT, smem, st>>>(a);
  return (int)cudaGetLastError();
}

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
