// me_proc_group.cu -- one translation unit per (process, precision) in the lane-group layout (me_group.cuh):
//   -DME_PROC=<name> -DME_PROC_UP=<NAME> -DME_PREC=<0|1|2> [-DME_MINB=<min amplitude warps per SM>]
// exports  me_launch_<name>_p<prec>  (C++ linkage, called from me_api.cu), same contract as me_proc.cu.
// A call runs the events in chunks that fit the handle's scratch; per chunk three kernels on the caller's stream:
// setup_kernel (K0) -> amp_kernel (K1) -> colour_kernel (K2).
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
#ifndef ME_NPART
#define ME_NPART 2   // parts of the scratch (me::PipeCtx holds 4 events for them); 2, 3 and 4 measured: 2 is best
#endif
#include <cstdio>
#include <cstdlib>

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

// colour-matrix numerators: integers of magnitude <= 4096 (exact in fp64, fp32 and TF32), read once per block of K2
__device__ const short c_cmat16[Grp::ncol * Grp::ncol] = ME_CAT(ME_CMAT_, ME_PROC_UP);
struct CMat {
  __device__ __forceinline__ static int at16(int i) { return (int)__ldg(c_cmat16 + i); }
};

// 120 flows: C' in MMA fragment order, written by cfrag_kernel at the start of every call (a few microseconds; no
// state to keep: concurrent calls write the same values)
__device__ T_col g_cfrag[me::ColGeom<Grp, T_col>::CF_GLOBAL ? me::ColGeom<Grp, T_col>::CF : 1];

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

template <int MODE, typename TA, typename TCo>
static int launch_mode(const me::LaunchArgs& a, cudaStream_t st, me::LaunchInfo* info, bool dry) {
  typedef me::GrpGeom<Grp, TA> GE;
  typedef me::ColGeom<Grp, TCo> CG;
  typedef me::GrpEvent<TA, Grp::n> EV;
  constexpr int N = Grp::n;
  auto k0 = me::setup_kernel<TA, N>;
  auto k1 = me::amp_kernel<Grp, TA, TCo, ME_MINB>;
  auto k2 = me::colour_kernel<Grp, TCo, CMat, MODE>;
  // the gluon-helicity combinations with at least one good helicity row
  me::PipeArgs p;
  memset(&p, 0, sizeof(p));
  for (int gg = 0; gg < GE::NGRP; gg++) {
    int m = 0;
    for (int v = 0; v < 4; v++) {
      const int h = me::grp_hel_of<N>(gg, v);
      if (MODE == me::MODE_FILTER || ((a.good.mask[h >> 6] >> (h & 63)) & 1ull)) m |= 1 << v;
    }
    if (m) { p.combo[p.ncombo] = (unsigned char)gg; p.vmask[p.ncombo] = (unsigned char)m; p.ncombo++; }
  }
  const size_t evb = sizeof(EV), grpb = (size_t)me::XGeom<Grp>::GRP * sizeof(TCo);
  const size_t per_event = evb + (size_t)p.ncombo * grpb, slack = 2 * grpb + 1024;
  const int nunit = (p.ncombo + GE::GPW - 1) / GE::GPW;
  // Chunks: the scratch is used as NPART parts in turn; with at least two chunks, consecutive chunks run on
  // alternating internal streams and the colour kernel of chunk c overlaps the amplitude kernels of later chunks.
  const int NPART = ME_NPART;
  const size_t half = (a.scratch_bytes / NPART) & ~(size_t)255;
  long long cap = (half > slack) ? (long long)((half - slack) / per_event) : 0;   // events per half
  if (cap > (1 << 20)) cap = 1 << 20;
  const long long min_chunk = (8 * 1184 + nunit - 1) / (nunit > 0 ? nunit : 1);   // >= 8 waves of amplitude warps on 148 SMs
  long long chunk = cap;
  if (chunk > 0 && a.nevt > 0) {
    long long want = (a.nevt + 2 * NPART - 1) / (2 * NPART);      // aim at two rounds of the parts per call
    if (want < min_chunk) want = min_chunk;
    if (want < chunk) chunk = want;
  }
  const long long nchunks = (chunk > 0) ? (a.nevt + chunk - 1) / chunk : 0;
  int dev = 0, sms = 0;
  cudaError_t err = cudaGetDevice(&dev);
  if (err == cudaSuccess) err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (err != cudaSuccess) return (int)err;
  if (info) {
    cudaFuncAttributes fa;
    err = cudaFuncGetAttributes(&fa, k1);
    if (err != cudaSuccess) return (int)err;
    info->threads = 32;
    info->blocks = (int)((a.nevt < chunk ? a.nevt : chunk) * nunit);
    info->regs = fa.numRegs;
    info->local_bytes = (int)fa.localSizeBytes;
    info->cum_slots = 0;
    info->scratch_per_event = (long long)(sizeof(EV) + (size_t)GE::NGRP * grpb);
    info->chunk = chunk;
    {  // what this batch would like to have: NPART parts of its preferred chunk (all combinations), whatever a.scratch_bytes is
      long long want = (a.nevt + 2 * NPART - 1) / (2 * NPART);
      if (want < min_chunk) want = min_chunk;
      if (want > a.nevt) want = a.nevt;
      if (want > (1 << 20)) want = 1 << 20;
      if (want < 1) want = 1;
      info->scratch_wanted = (long long)NPART * (long long)(align_up((size_t)want * (size_t)info->scratch_per_event + slack, 256) + 256);
    }
    info->launches = (int)(3 * nchunks) + (CG::CF_GLOBAL ? 1 : 0);
  }
  if (dry || a.nevt == 0) return 0;
  if (p.ncombo == 0 || chunk < 1 || !a.scratch) return (int)cudaErrorInvalidValue;
  // Once per device (not per call: a 256-event step is a few tens of microseconds): the kernels' shared-memory limits
  // and the colour kernel's residency.  Shared memory of K1: what ME_MINB amplitude warps need and no more (the rest of
  // the 256 KB stays L1 for the table words).
  constexpr int k1_smem = GE::SMEM;
  static int k2_cached[64];   // colour-kernel blocks per SM on each device ordinal, 0 = not set up yet
  if (dev < 0 || dev >= 64) return (int)cudaErrorInvalidDevice;
  int k2_per_sm = k2_cached[dev];
  if (k2_per_sm == 0) {
    int carve = (int)((size_t)ME_MINB * (GE::SMEM + 1024) * 100 / (228 * 1024)) + 1;
    if (carve > 100) carve = 100;
    err = cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, k1_smem);
    if (err == cudaSuccess) err = cudaFuncSetAttribute(k1, cudaFuncAttributePreferredSharedMemoryCarveout, carve);
    if (err == cudaSuccess) err = cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, CG::SMEM);
    if (err == cudaSuccess) err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&k2_per_sm, k2, CG::WARPS * 32, CG::SMEM);
    if (err != cudaSuccess) return (int)err;
    if (k2_per_sm < 1) k2_per_sm = 1;
    k2_cached[dev] = k2_per_sm;   // same value from every thread that gets here first
  }
  if (CG::CF_GLOBAL) {
    void* sym = nullptr;
    static_assert(sizeof(TCo) == sizeof(T_col), "the filter (fp64) is compiled in the fp64 unit only");
    err = cudaGetSymbolAddress(&sym, g_cfrag);
    if (err != cudaSuccess) return (int)err;
    me::cfrag_kernel<Grp, TCo, CMat><<<(CG::CF + 255) / 256, 256, 0, st>>>((TCo*)sym);
    p.cfrag = sym;
  }
  const me::PipeCtx* px = (nchunks > 1) ? a.pipe : nullptr;
  if (px) {  // fork: the internal streams start after everything already enqueued on the caller's stream
    err = cudaEventRecord(px->fork, st);
    if (err == cudaSuccess) err = cudaStreamWaitEvent(px->sa, px->fork, 0);
    if (err == cudaSuccess) err = cudaStreamWaitEvent(px->sb, px->fork, 0);
    if (err == cudaSuccess) err = cudaStreamWaitEvent(px->s2, px->fork, 0);
    if (err != cudaSuccess) return (int)err;
  }
  long long c = 0;
  for (long long e0 = 0; e0 < a.nevt; e0 += chunk, c++) {
    const long long n = (a.nevt - e0 < chunk) ? (a.nevt - e0) : chunk;
    const int hf = (int)(c & 1), part = (int)(c % NPART);
    char* base = (char*)a.scratch + (px ? (size_t)part * half : 0);
    p.a = a;
    p.a.nevt = n;
    p.a.mom = a.mom + e0 * (Grp::npar * 4);
    p.a.gs = a.gs + e0;
    p.a.rndhel = a.rndhel ? a.rndhel + e0 : nullptr;
    p.a.rndcol = a.rndcol ? a.rndcol + e0 : nullptr;
    p.a.me = a.me ? a.me + e0 : nullptr;
    p.a.selhel = a.selhel ? a.selhel + e0 : nullptr;
    p.a.selcol = a.selcol ? a.selcol + e0 : nullptr;
    p.a.channel = a.channel ? a.channel + e0 : nullptr;   // multichannel: the colour kernel indexes it with the chunk-local event
    p.ev = base;
    p.xt = base + align_up((size_t)n * evb, 256);
    constexpr int PT = ((1 << N) + N + 6 <= 32) ? 32 : 64;
    cudaStream_t s1 = px ? (hf ? px->sb : px->sa) : st, s2 = px ? px->s2 : st;
#ifdef ME_K2_SAME_STREAM
    // units for which it measured faster (build.py): the colour kernel follows the amplitude kernel of its chunk on the same
    // low-priority stream instead of cutting in on the high-priority one (no SM is drained for it ahead of time)
    s2 = s1;
#endif
    if (px && c >= NPART && (err = cudaStreamWaitEvent(s1, px->k2[part], 0)) != cudaSuccess) return (int)err;  // part free again
#if defined(ME_CHECK) && ME_CHECK
    // self-check build: the part of the scratch this chunk uses starts as NaN
    if ((err = cudaMemsetAsync(base, 0xff, align_up((size_t)n * evb, 256) + (size_t)n * p.ncombo * grpb + slack, s1)) != cudaSuccess) return (int)err;
#endif
    k0<<<(unsigned)((n * PT + 127) / 128), 128, 0, s1>>>(p.a, (EV*)p.ev);
    k1<<<(unsigned)(n * nunit), 32, k1_smem, s1>>>(p);
    if (px) {
      if ((err = cudaEventRecord(px->k1[hf], s1)) != cudaSuccess) return (int)err;
      if ((err = cudaStreamWaitEvent(s2, px->k1[hf], 0)) != cudaSuccess) return (int)err;
    }
    // colour kernel: WPS warps per SM (or one warp per event if that is fewer); the warps stride over the events
    long long b2 = (n + CG::WARPS - 1) / CG::WARPS;
    long long cap2 = (long long)sms * ((CG::WPS + CG::WARPS - 1) / CG::WARPS);
    if (cap2 > (long long)sms * k2_per_sm) cap2 = (long long)sms * k2_per_sm;
    if (b2 > cap2) b2 = cap2;
    k2<<<(unsigned)b2, CG::WARPS * 32, CG::SMEM, s2>>>(p);
    if (px && (err = cudaEventRecord(px->k2[part], s2)) != cudaSuccess) return (int)err;
    err = cudaGetLastError();
    if (err != cudaSuccess) return (int)err;
  }
  if (px) {  // join: the caller's stream continues after the last colour kernel (s2 is in order, and follows sa / sb)
    err = cudaStreamWaitEvent(st, px->k2[(int)((c - 1) % NPART)], 0);
    if (err != cudaSuccess) return (int)err;
#ifdef ME_K2_SAME_STREAM
    // the colour kernels of the last two chunks ran on different streams: wait for both
    if (c >= 2 && (err = cudaStreamWaitEvent(st, px->k2[(int)((c - 2) % NPART)], 0)) != cudaSuccess) return (int)err;
#endif
  }
  return 0;
}

// mode: me::MODE_*; dry = only report the launch geometry in *info.
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
