// me_kernels.cuh -- the event kernel (layout "B0": one event per thread, helicity loop inside).
//
// Hot path of SURVEY.md 8(a): a1 load (coalesced tile -> shared memory -> registers), a2-a5 generated
// amplitude code (csrc/gen/proc_*.cuh), a6 colour quadratic form, a7 helicity loop over the good
// helicities, a8 helicity/colour selection, a9 store.  "event-level data parallelism ... lockstep
// processing": every thread of a warp runs the same straight-line code on its own event.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "me_ops.cuh"
#include "me_params.cuh"

namespace me {


struct GoodList {
  int n;
  uint8_t h[128];               // good helicity rows in increasing order
  unsigned long long mask[2];   // the same as a bit mask (bit h of mask[h >> 6])
};

struct LaunchArgs {
  const double* mom;
  const double* gs;
  const double* rndhel;
  const double* rndcol;
  long long nevt;
  double* me;
  int* selhel;
  int* selcol;
  double* cum;                 // scratch [ngood][nslots] running helicity sums (selection only)
  unsigned long long* fracmax; // filter: [ncomb] max over events of |M_h|^2 / sum (bit pattern of a double)
  int blocks;                  // 0 = choose
  void* scratch;               // lane-group pipeline: per-event data and jamps between its kernels (owned by the handle)
  size_t scratch_bytes;
  const struct PipeCtx* pipe;  // lane-group pipeline: the handle's internal streams and events (host side only)
  const int* channel;          // multichannel: [nevt] channel (diagram) of every event, or nullptr
  int nchan;                   // multichannel: number of channels (channel ids are clamped to 0 .. nchan-1)
  const unsigned* chanflows;   // multichannel: [nchan][4] bit c set iff colour flow c is allowed for the channel
  DevParams par;
  GoodList good;
};

// Internal streams of a handle (lane-group pipeline): consecutive chunks of events alternate between sa and sb
// (setup + amplitude kernels) so that the tail of one chunk's amplitude kernel is filled by the next chunk's, and
// every colour kernel runs on the high-priority stream s2 beside the amplitude kernel of the following chunk.
struct PipeCtx {
  cudaStream_t sa, sb, s2;
  cudaEvent_t fork, k1[2], k2[4];
};

struct LaunchInfo {
  int threads, blocks, regs, local_bytes;   // of the dominant (amplitude) kernel
  long long cum_slots;          // one-event-per-thread kernel, MODE_SELECT scratch: doubles per good helicity
  long long scratch_per_event;  // lane-group pipeline: scratch bytes per event of a chunk (0: not used)
  long long chunk;              // lane-group pipeline: events per chunk with the scratch given
  long long scratch_wanted;     // lane-group pipeline: scratch bytes with which a call of a.nevt events runs in its preferred chunks
  int launches;                 // kernels enqueued by the call
};

enum { MODE_ME = 0, MODE_SELECT = 1, MODE_FILTER = 2 };

// colour quadratic form  sum_ab C_ab (Re J_a Re J_b + Im J_a Im J_b)  using the symmetry of C:
//   = sum_a [ C_aa |J_a|^2 + 2 Re( conj(J_a) sum_{b>a} C_ab J_b ) ],   C given as integers / cden
//   CM::at(i): entry i of the row-major integer numerator matrix, held as TC in constant memory
template <int NCOL, typename TC, typename TJ, class CM>
__device__ __forceinline__ TC colour_sum(const cx<TJ>* J) {
  TC s = TC(0);
  if (NCOL <= 24) {
#pragma unroll
    for (int a = 0; a < NCOL; a++) {
      const TC are = TC(J[a].re), aim = TC(J[a].im);
      TC yre = TC(0.5) * CM::at(a * NCOL + a) * are, yim = TC(0.5) * CM::at(a * NCOL + a) * aim;
#pragma unroll
      for (int b = a + 1; b < NCOL; b++) {
        yre += CM::at(a * NCOL + b) * TC(J[b].re);
        yim += CM::at(a * NCOL + b) * TC(J[b].im);
      }
      s += are * yre + aim * yim;
    }
  } else {
    for (int a = 0; a < NCOL; a++) {
      const TC are = TC(J[a].re), aim = TC(J[a].im);
      TC yre = TC(0.5) * CM::at(a * NCOL + a) * are, yim = TC(0.5) * CM::at(a * NCOL + a) * aim;
#pragma unroll 8
      for (int b = a + 1; b < NCOL; b++) {
        yre += CM::at(a * NCOL + b) * TC(J[b].re);
        yim += CM::at(a * NCOL + b) * TC(J[b].im);
      }
      s += are * yre + aim * yim;
    }
  }
  return TC(2) * s;
}

template <int N> __device__ __forceinline__ double ipow(double g) {
  double r = 1.0;
#pragma unroll
  for (int i = 0; i < N; i++) r *= g;
  return r;
}

// P: generated process struct; T: amplitude arithmetic; TC: colour-sum arithmetic; CM: constant colour matrix
template <class P, typename T, typename TC, class CM, int MODE, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) event_kernel(const LaunchArgs a) {
  constexpr int NP4 = P::npar * 4;
  constexpr int STR = NP4 + 1;  // odd stride: conflict-free per-thread reads
  __shared__ double smom[NT * STR];
  const long long ntiles = (a.nevt + NT - 1) / NT;
  const int slot = blockIdx.x * NT + threadIdx.x;
  const long long nslots = (long long)gridDim.x * NT;
  for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const long long e0 = tile * NT;
    const long long nhere = (a.nevt - e0 < NT) ? (a.nevt - e0) : NT;
    __syncthreads();
    // a1: the tile's momenta are one contiguous block of nhere*npar*4 doubles: coalesced load
    for (int i = threadIdx.x; i < nhere * NP4; i += NT) smom[(i / NP4) * STR + (i % NP4)] = a.mom[e0 * NP4 + i];
    __syncthreads();
    const long long e = e0 + threadIdx.x;
    if (e >= a.nevt) continue;
    typename P::template Event<T> ev;
    const double* pm = smom + threadIdx.x * STR;
    P::template setup<T>([pm](int i, int m) { return pm[4 * i + m]; }, a.par, ev);
    double total = 0.0;
    TC wc[(MODE == MODE_SELECT) ? P::ncol : 1];
    if (MODE == MODE_SELECT) {
#pragma unroll
      for (int c = 0; c < P::ncol; c++) wc[c] = TC(0);
    }
    const int nh = (MODE == MODE_FILTER) ? P::ncomb : a.good.n;
    double mh_all[(MODE == MODE_FILTER) ? P::ncomb : 1];
#pragma unroll 1
    for (int ih = 0; ih < nh; ih++) {
      const int h = (MODE == MODE_FILTER) ? ih : a.good.h[ih];
      cx<T> J[P::ncol];
      P::template jamps<T>(ev, h, J);
      const double mh = (double)colour_sum<P::ncol, TC, T, CM>(J);
      total += mh;
      if (MODE == MODE_SELECT) {
        a.cum[(long long)ih * nslots + slot] = total;
#pragma unroll
        for (int c = 0; c < P::ncol; c++) wc[c] += TC(J[c].re) * TC(J[c].re) + TC(J[c].im) * TC(J[c].im);
      }
      if (MODE == MODE_FILTER) mh_all[ih] = mh;
    }
    if (MODE == MODE_FILTER) {
      for (int ih = 0; ih < P::ncomb; ih++) {
        const double f = (total > 0.0) ? mh_all[ih] / total : 0.0;
        atomicMax(a.fracmax + ih, (unsigned long long)__double_as_longlong(f));
      }
      continue;
    }
    const double g = P::ngl ? a.gs[e] : 1.0;
    a.me[e] = total * ipow<2 * P::ngl>(g) * (1.0 / (double(P::denom) * double(P::cden)));
    if (MODE == MODE_SELECT) {
      if (a.selhel) {
        const double target = a.rndhel[e] * total;
        int sel = a.good.h[nh - 1];
        for (int ih = 0; ih < nh; ih++)
          if (target < a.cum[(long long)ih * nslots + slot]) { sel = a.good.h[ih]; break; }
        a.selhel[e] = sel;
      }
      if (a.selcol) {
        // multichannel (reading R17): flows the event's channel does not contribute to get weight zero
        const unsigned* cfl = a.channel ? a.chanflows + 4 * min(max(a.channel[e], 0), a.nchan - 1) : nullptr;
        auto allowed = [&](int c) { return !cfl || ((cfl[c >> 5] >> (c & 31)) & 1u); };
        double tot = 0.0;
#pragma unroll
        for (int c = 0; c < P::ncol; c++) tot += allowed(c) ? (double)wc[c] : 0.0;
        const double target = a.rndcol[e] * tot;
        int sel = P::ncol - 1;
        double run = 0.0;
        bool found = false;
#pragma unroll
        for (int c = 0; c < P::ncol; c++) {
          if (allowed(c)) {
            run += (double)wc[c];
            if (!found) { sel = c; found = target < run; }   // ends on the first hit, else on the last allowed flow
          }
        }
        a.selcol[e] = sel;
      }
    }
  }
}

}  // namespace me
