// me_diag.cuh -- the diagram-by-diagram kernel: single-diagram-enhancement weights for multichannel running
// ("events from different channels" in one launch; reading R17).
//
//   num[e] = sum_{h good} sum_{terms t of diagram d = channel[e]} |A_{d,t}(h)|^2      den[e] = the same over ALL diagrams
//
// A_{d,t} is the value of ONE Feynman diagram (one colour-structure term of it if it has four-gluon vertices).  The
// matrix-element kernels never form single diagrams (they sum colour-ordered currents), so this quantity has its own
// kernel, fp64 whatever the build.  One BLOCK per event; per good helicity the block evaluates, level by level from
// the generated tables (codegen/emit_diag.py), every gluon tree once (shared by the diagrams that contain it), every
// quark-line prefix once, then every closure, with the phase-stripped rules of me_ops.cuh (the stripped factors have
// modulus one, and every diagram carries g_s^n, applied at the end).  Tree currents and prefixes live in shared
// memory; the helicity-independent event data are the GrpEvent<double, n> made by setup_kernel.
// A warp never mixes channels by construction: the channel only selects which closures also count for num.
#pragma once
#include "me_group.cuh"

namespace me {

struct DiagArgs {
  LaunchArgs a;              // mom, gs, nevt, good (list of good helicity rows), par
  const void* ev;            // GrpEvent<double, n>[nevt]
  const int* channel;        // [nevt] or nullptr (then num is not written)
  double* num;               // [nevt] or nullptr
  double* den;               // [nevt]
};

template <class D> struct DiagGeom {
  // Threads per event.  The levels of gg -> t tbar g g hold 6 .. 45 tasks (159 closures): one warp wastes a quarter of
  // its thread slots there, four warps two thirds, and wait at eight barriers per helicity (ncu, round 3: barrier stall
  // 7.5 per issued instruction with 128 threads).  Five gluons have levels of 10 .. 510 tasks and 1890 closures.
#ifndef ME_DIAG_NT4
#define ME_DIAG_NT4 32    // threads per event for four gluons (32 / 64 / 128 measured: 25.3 / 28.2 / 34.5 ms per 65536 events)
#endif
#ifndef ME_DIAG_NT5
#define ME_DIAG_NT5 256   // threads per event for five gluons (145 KB of slots: one block per SM; 64 / 128 / 256 / 512 / 1024
                          // threads measured: 56.9 / 37.5 / 33.6 / 33.7 / 43.6 ms per 4096 events)
#endif
  static constexpr int NT = (D::n >= 5) ? ME_DIAG_NT5 : ((D::n == 4) ? ME_DIAG_NT4 : 32);
  // A slot (4 complex doubles) takes SS = 10 doubles: with 80-byte strides the 16-byte accesses of eight neighbouring
  // slots fall into eight different bank groups (with 64-byte strides they met four to a group: 3.8e9 bank conflicts
  // on 2.3e9 ideal wavefronts in the same capture)
  static constexpr int SS = 10;
  static constexpr int EVB = (((int)sizeof(GrpEvent<double, D::n>) + 127) / 128) * 128;
  static constexpr int SMEM = EVB + (D::ntree + D::nnode) * SS * 8;   // event data, tree currents, quark-line prefixes
};

template <class D>
__global__ void __launch_bounds__(DiagGeom<D>::NT) diag_kernel(const DiagArgs p) {
  constexpr int N = D::n, NPAR = N + 2, NT = DiagGeom<D>::NT, SS = DiagGeom<D>::SS;
  typedef GrpEvent<double, N> EV;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  EV& ev = *reinterpret_cast<EV*>(smem_raw);
  double* trees = reinterpret_cast<double*>(smem_raw + DiagGeom<D>::EVB);
  double* chain = trees + D::ntree * SS;
  __shared__ double red[2][NT / 32];
  const int tid = threadIdx.x;
  const LaunchArgs& a = p.a;
  for (long long e = blockIdx.x; e < a.nevt; e += gridDim.x) {
    __syncthreads();
    {
      const int4* src = reinterpret_cast<const int4*>(reinterpret_cast<const EV*>(p.ev) + e);
      int4* dst = reinterpret_cast<int4*>(&ev);
      for (int i = tid; i < (int)(sizeof(EV) / 16); i += NT) dst[i] = __ldcg(src + i);
    }
    const int mych = p.channel ? p.channel[e] : -1;
    double num = 0.0, den = 0.0;
#pragma unroll 1
    for (int ih = 0; ih < a.good.n; ih++) {
      const int h = a.good.h[ih];
      __syncthreads();   // event data staged / the closures of the previous helicity are done with the shared arrays
      // leaves: polarisation vectors of this helicity row; root of the quark line
      if (tid < N) {
        const int pp = (tid < 2) ? tid : tid + 2;
        const int lam = ((h >> (NPAR - 1 - pp)) & 1) ? 1 : -1;
        polbasis<double> pb;
        for (int c = 0; c < 3; c++) { pb.e1[c] = ev.pol[tid][c]; pb.e2[c] = ev.pol[tid][3 + c]; }
        GrpVec<double>::st(trees + tid * SS, polvec(pb, lam, pp >= 2));
      }
      if (tid == N) {
        const int ht = (h >> (NPAR - 1 - 2)) & 1;
        for (int c = 0; c < 8; c++) chain[c] = ev.ub[ht][c];
      }
      const int htb = (h >> (NPAR - 1 - 3)) & 1;
      __syncthreads();
      // gluon trees by number of legs
#pragma unroll 1
      for (int L = 2; L <= N; L++) {
        for (int t = D::tree_off(L - 2) + tid; t < D::tree_off(L - 1); t += NT) {
          const unsigned* w = D::tree() + 4 * t;
          const unsigned w0 = __ldg(w), w1 = __ldg(w + 1), w2 = __ldg(w + 2), w3 = __ldg(w + 3);
          const vec4<double> A = GrpVec<double>::ld(trees + (w1 & 0xffffu) * SS, 0u);
          const vec4<double> B = GrpVec<double>::ld(trees + (w1 >> 16) * SS, 0u);
          const double ik = ev.ik[w2 >> 16];
          vec4<double> J;
          if (((w0 >> 16) & 15u) == 0u) {
            mom4<double> kA, kB;
            for (int c = 0; c < 4; c++) { kA.c[c] = ev.Ksub[w3 & 255u][c]; kB.c[c] = ev.Ksub[(w3 >> 8) & 255u][c]; }
            J = vvv_current(A, B, kA, kB, ik);
          } else {
            const vec4<double> C = GrpVec<double>::ld(trees + (w2 & 0xffffu) * SS, 0u);
            vec4<double> J0, J1, J2;
            vvvv_currents(A, B, C, ik, J0, J1, J2);
            const unsigned term = (w0 >> 20) & 3u;
            J = (term == 0u) ? J0 : ((term == 1u) ? J1 : J2);
          }
          GrpVec<double>::st(trees + (w0 & 0xffffu) * SS, J);
        }
        __syncthreads();
      }
      // quark-line prefixes by number of attached trees
#pragma unroll 1
      for (int d = 0; d < D::nchainlev; d++) {
        for (int t = D::chain_off(d) + tid; t < D::chain_off(d + 1); t += NT) {
          const unsigned w0 = __ldg(D::chain() + 2 * t), w1 = __ldg(D::chain() + 2 * t + 1);
          const spin4<double> R = ld_spin<double>(chain + (w0 >> 16) * SS);
          const vec4<double> J = GrpVec<double>::ld(trees + (w1 & 0xffffu) * SS, 0u);
          const unsigned m = w1 >> 16;
          mom4<double> q;
          for (int c = 0; c < 4; c++) q.c[c] = ev.qsub[m][c];
          const spin4<double> X = row_prop(row_slash(R, J), q, ev.mt, mk<double>(ev.gd[m][0], ev.gd[m][1]));
          vec4<double> o;
          for (int c = 0; c < 4; c++) o.c[c] = X.c[c];
          GrpVec<double>::st(chain + (w0 & 0xffffu) * SS, o);
        }
        __syncthreads();
      }
      // closures
      const spin4<double> vv = ld_spin<double>(ev.v[htb]);
      for (int t = tid; t < D::nclos; t += NT) {
        const unsigned w0 = __ldg(D::clos() + 2 * t), ch = __ldg(D::clos() + 2 * t + 1);
        const spin4<double> R = ld_spin<double>(chain + (w0 & 0xffffu) * SS);
        const vec4<double> J = GrpVec<double>::ld(trees + (w0 >> 16) * SS, 0u);
        const double a2 = norm2(row_col(row_slash(R, J), vv));
        den += a2;
        num += ((int)ch == mych) ? a2 : 0.0;
      }
    }
    // block sums in a fixed order (bit-reproducible), then g_s^(2n)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      num += __shfl_xor_sync(0xffffffffu, num, o);
      den += __shfl_xor_sync(0xffffffffu, den, o);
    }
    if ((tid & 31) == 0) { red[0][tid >> 5] = num; red[1][tid >> 5] = den; }
    __syncthreads();
    if (tid == 0) {
      double sn = 0.0, sd = 0.0;
      for (int w = 0; w < NT / 32; w++) { sn += red[0][w]; sd += red[1][w]; }
      const double g = ipow<2 * N>(a.gs[e]);
      if (p.num && p.channel) p.num[e] = sn * g;
      p.den[e] = sd * g;
    }
  }
}

}  // namespace me
