// me_group.cuh -- the "lane-group" event kernel (layout B2) for g g -> t tbar + (n-2) g, n >= 4.
//
// One CUDA block per event.  A GROUP of LPG lanes of one warp owns one combination of the n gluon helicities
// (n = 4: 4 lanes, one per first gluon s1 of the colour flow, both t helicities walked by the same lane; n = 5:
// 10 lanes (s1, h_t)); the four (h_t, h_tbar) combinations are handled inside the group, so the gluon currents
// are computed once per gluon-helicity combination instead of once per helicity.
// Per event the block first forms the helicity-independent data in shared memory (one branch-free phase, one
// block barrier); then every group runs, warp-synchronously:
//   leaves  lane i < n      : polarisation vector of gluon i (a2)                       -> shared memory slot
//   tree    lane = sequence : colour-ordered currents Jord(seq), |seq| = 2..n-1 (a3)    -> shared memory slot
//           |seq| = n       : contracted at once with the four t-tbar currents Q(h_t,h_tbar) -> J init (a4, a5)
//   walk    lane = s1       : quark line for the flows that start with gluon s1 (a3-a5) -> J[flow][h_t][h_tbar]
//   colour  task = (h_t,h_tbar[,re/im]): x^T C x over the n! flows (a6)                 -> |M_h|^2
// and one warp sums the good helicities in table order (a7), selects helicity / colour (a8) and stores (a9).
// Current operands of the walk are read from shared memory with 16-byte loads (the lanes of a quarter-warp read
// different slots: chunk-swizzled in the fp64 build) and feed both t helicities; the running spinors stay in
// registers.  fp32 build: the two t-helicity chains, the complex arithmetic of the tree vertices and the colour
// sum are packed f32x2 operations (FFMA2).  DESIGN.md section 5 has the measured history of these choices.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "me_kernels.cuh"

namespace me {

// Packed pair of floats: lane-local SIMD over the two t helicities of the quark-line walk in the fp32 build
// (sm_100a FFMA2 / FMUL2 / FADD2: two fp32 operations per issued instruction; negation and the broadcast of a
// scalar are operand modifiers, so make_float2(-x,-y) and make_float2(x,x) cost nothing).
struct f2 {
  float2 v;
};
__device__ __forceinline__ f2 mkf2(float x, float y) { f2 r; r.v = make_float2(x, y); return r; }
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { f2 r; r.v = __fadd2_rn(a.v, b.v); return r; }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { f2 r; r.v = __fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y)); return r; }
__device__ __forceinline__ f2 operator-(f2 a) { return mkf2(-a.v.x, -a.v.y); }
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { f2 r; r.v = __fmul2_rn(a.v, b.v); return r; }
__device__ __forceinline__ f2 fmad(f2 a, f2 b, f2 c) { f2 r; r.v = __ffma2_rn(a.v, b.v, c.v); return r; }

// How the walk keeps the t helicities of a lane: NCH register chains of scalar type PS
template <typename T, bool HTL> struct WalkPack {
  typedef T PS;
  static constexpr int NCH = HTL ? 2 : 1;
  __device__ __forceinline__ static PS widen(T x) { return x; }
};
template <> struct WalkPack<float, true> {
  typedef f2 PS;
  static constexpr int NCH = 1;
  __device__ __forceinline__ static PS widen(float x) { return mkf2(x, x); }
};

template <typename T, typename TC, int N>
struct alignas(16) GrpEvent {
  double mh[1 << (N + 2)];     // |M_h|^2 (colour-summed, un-normalised) per helicity row
  alignas(16) T Ksub[1 << N][4];           // sum of the gluon momenta of a subset (bit i = gluon i)
  alignas(16) T qsub[1 << N][4];           // -(k_t + K_S): momentum of the quark line after the gluons of S
  T gd[1 << N][2];             // 1 / (q^2 - m^2 + i m Gamma)
  T ik[1 << N];                // 1 / K_S^2
  alignas(16) T Q[4][8];                   // ubar(h_t) gamma^mu v(h_tbar), index 2 h_t + h_tbar
  alignas(16) T ub[2][8];
  alignas(16) T v[2][8];
  T pol[N][6];
  T mt;
  TC wc[5][(N == 4) ? 24 : (N == 5 ? 120 : 6)];  // per-warp colour weights (at most 4 warps per block)
  unsigned char gmask[1 << N];  // per gluon-helicity combination: bit v set iff helicity row (combination, v) is good
};

template <typename T> struct GrpVec;
template <> struct GrpVec<double> {
  __device__ __forceinline__ static vec4<double> ld(const double* p, unsigned neg) {
    vec4<double> r;
    const double2* q = reinterpret_cast<const double2*>(p);
    const int m = (int)(neg << 31);
#pragma unroll
    for (int i = 0; i < 4; i++) {
      const double2 x = q[i];
      r.c[i].re = __hiloint2double(__double2hiint(x.x) ^ m, __double2loint(x.x));
      r.c[i].im = __hiloint2double(__double2hiint(x.y) ^ m, __double2loint(x.y));
    }
    return r;
  }
  __device__ __forceinline__ static void st(double* p, const vec4<double>& a) {
    double2* q = reinterpret_cast<double2*>(p);
#pragma unroll
    for (int i = 0; i < 4; i++) q[i] = make_double2(a.c[i].re, a.c[i].im);
  }
};
template <> struct GrpVec<float> {
  __device__ __forceinline__ static vec4<float> ld(const float* p, unsigned neg) {
    vec4<float> r;
    const float4* q = reinterpret_cast<const float4*>(p);
    const int m = (int)(neg << 31);
#pragma unroll
    for (int i = 0; i < 2; i++) {
      const float4 x = q[i];
      r.c[2 * i].re = __int_as_float(__float_as_int(x.x) ^ m);
      r.c[2 * i].im = __int_as_float(__float_as_int(x.y) ^ m);
      r.c[2 * i + 1].re = __int_as_float(__float_as_int(x.z) ^ m);
      r.c[2 * i + 1].im = __int_as_float(__float_as_int(x.w) ^ m);
    }
    return r;
  }
  __device__ __forceinline__ static void st(float* p, const vec4<float>& a) {
    float4* q = reinterpret_cast<float4*>(p);
#pragma unroll
    for (int i = 0; i < 2; i++) q[i] = make_float4(a.c[2 * i].re, a.c[2 * i].im, a.c[2 * i + 1].re, a.c[2 * i + 1].im);
  }
};

template <typename T> __device__ __forceinline__ spin4<T> ld_spin(const T* p) {
  const vec4<T> x = GrpVec<T>::ld(p, 0u);
  spin4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) r.c[i] = x.c[i];
  return r;
}

// Current slots (8 T = 64 or 32 bytes each) are stored with their 16-byte chunks permuted by the slot index
// (chunk i of slot s sits at position i ^ x(s)), so that the slots the lanes of a quarter-warp read together fall
// into different bank groups: without it a 64-byte slot stride reaches only half of the banks for a given chunk.
template <typename T> struct GrpSlot;
template <> struct GrpSlot<double> {
  __device__ __forceinline__ static vec4<double> ld(const double* slots, unsigned s, unsigned neg) {
    const char* base = reinterpret_cast<const char*>(slots + s * 8);
    const unsigned x = (s >> 1) & 3u;
    const int m = (int)(neg << 31);
    vec4<double> r;
#pragma unroll
    for (int i = 0; i < 4; i++) {
      const double2 v = *reinterpret_cast<const double2*>(base + ((i ^ x) << 4));
      r.c[i].re = __hiloint2double(__double2hiint(v.x) ^ m, __double2loint(v.x));
      r.c[i].im = __hiloint2double(__double2hiint(v.y) ^ m, __double2loint(v.y));
    }
    return r;
  }
  __device__ __forceinline__ static void st(double* slots, unsigned s, const vec4<double>& a) {
    char* base = reinterpret_cast<char*>(slots + s * 8);
    const unsigned x = (s >> 1) & 3u;
#pragma unroll
    for (int i = 0; i < 4; i++) *reinterpret_cast<double2*>(base + ((i ^ x) << 4)) = make_double2(a.c[i].re, a.c[i].im);
  }
};
template <> struct GrpSlot<float> {
  __device__ __forceinline__ static vec4<float> ld(const float* slots, unsigned s, unsigned neg) {
    const char* base = reinterpret_cast<const char*>(slots + s * 8);
    const unsigned x = 0u;  // fp32: the extra address arithmetic costs more issue slots than the conflicts (measured)
    const int m = (int)(neg << 31);
    vec4<float> r;
#pragma unroll
    for (int i = 0; i < 2; i++) {
      const float4 v = *reinterpret_cast<const float4*>(base + ((i ^ x) << 4));
      r.c[2 * i].re = __int_as_float(__float_as_int(v.x) ^ m);
      r.c[2 * i].im = __int_as_float(__float_as_int(v.y) ^ m);
      r.c[2 * i + 1].re = __int_as_float(__float_as_int(v.z) ^ m);
      r.c[2 * i + 1].im = __int_as_float(__float_as_int(v.w) ^ m);
    }
    return r;
  }
  __device__ __forceinline__ static void st(float* slots, unsigned s, const vec4<float>& a) {
    char* base = reinterpret_cast<char*>(slots + s * 8);
    const unsigned x = 0u;
#pragma unroll
    for (int i = 0; i < 2; i++)
      *reinterpret_cast<float4*>(base + ((i ^ x) << 4)) = make_float4(a.c[2 * i].re, a.c[2 * i].im, a.c[2 * i + 1].re, a.c[2 * i + 1].im);
  }
};

// acc += (A.B)(kA-kB) + ((kA+2kB).A) B - ((2kA+kB).B) A      (three-gluon vertex, propagator applied later)
template <typename T>
__device__ __forceinline__ void v3_acc(vec4<T>& acc, const vec4<T>& A, const vec4<T>& B, const T* kA, const T* kB) {
  const cx<T> ab = mdot(A, B);
  mom4<T> kab, k1, k2;
#pragma unroll
  for (int i = 0; i < 4; i++) {
    kab.c[i] = kA[i] - kB[i];
    k1.c[i] = kA[i] + T(2) * kB[i];
    k2.c[i] = -(T(2) * kA[i] + kB[i]);
  }
  const cx<T> ca = mdot(k1, A), cb = mdot(k2, B);
#pragma unroll
  for (int i = 0; i < 4; i++) {
    cx<T> t = fma(kab.c[i], ab, acc.c[i]);
    t = fma(ca, B.c[i], t);
    acc.c[i] = fma(cb, A.c[i], t);
  }
}
// acc += 2 (A.C) B - (B.C) A - (A.B) C       (colour-ordered four-gluon vertex)
template <typename T>
__device__ __forceinline__ void v4_acc(vec4<T>& acc, const vec4<T>& A, const vec4<T>& B, const vec4<T>& C) {
  const cx<T> ac = T(2) * mdot(A, C), bc = -mdot(B, C), ab = -mdot(A, B);
#pragma unroll
  for (int i = 0; i < 4; i++) {
    cx<T> t = fma(ac, B.c[i], acc.c[i]);
    t = fma(bc, A.c[i], t);
    acc.c[i] = fma(ab, C.c[i], t);
  }
}

// fp32 build: the same two vertices with every complex number as one packed f32x2 register pair (re, im): a complex
// multiply-add is two FFMA2 (the second with the operand halves swapped and one sign flipped, both operand
// modifiers on sm_100a) instead of four FFMA.
__device__ __forceinline__ float2 pk(const cx<float>& a) { return make_float2(a.re, a.im); }
__device__ __forceinline__ float2 cmul2(float2 a, float2 b) {  // a * b
  const float2 t = __fmul2_rn(make_float2(a.x, a.x), b);
  return __ffma2_rn(make_float2(-a.y, a.y), make_float2(b.y, b.x), t);
}
__device__ __forceinline__ float2 cmac2(float2 acc, float2 a, float2 b) {  // acc + a * b
  acc = __ffma2_rn(make_float2(a.x, a.x), b, acc);
  return __ffma2_rn(make_float2(-a.y, a.y), make_float2(b.y, b.x), acc);
}
__device__ __forceinline__ float2 cmsc2(float2 acc, float2 a, float2 b) {  // acc - a * b
  acc = __ffma2_rn(make_float2(-a.x, -a.x), b, acc);
  return __ffma2_rn(make_float2(a.y, -a.y), make_float2(b.y, b.x), acc);
}
__device__ __forceinline__ float2 rmac2(float2 acc, float s, float2 b) { return __ffma2_rn(make_float2(s, s), b, acc); }
// Minkowski product of two complex vectors / of a real and a complex vector.  Both factors vary from term to term
// here, so the second FFMA2 takes the broadcast of a.im (free) against (-b.im, b.re) (one sign flip) rather than a
// materialised (-a.im, a.im) pair (two moves).
__device__ __forceinline__ float2 mdot2(const float2 (&A)[4], const float2 (&B)[4]) {
  float2 r = __fmul2_rn(make_float2(A[0].x, A[0].x), B[0]);
  r = __ffma2_rn(make_float2(A[0].y, A[0].y), make_float2(-B[0].y, B[0].x), r);
#pragma unroll
  for (int i = 1; i < 4; i++) {
    r = __ffma2_rn(make_float2(-A[i].x, -A[i].x), B[i], r);
    r = __ffma2_rn(make_float2(A[i].y, A[i].y), make_float2(B[i].y, -B[i].x), r);
  }
  return r;
}
__device__ __forceinline__ float2 mdot2(const float (&k)[4], const float2 (&A)[4]) {
  float2 r = __fmul2_rn(make_float2(k[0], k[0]), A[0]);
  r = rmac2(r, -k[1], A[1]);
  r = rmac2(r, -k[2], A[2]);
  return rmac2(r, -k[3], A[3]);
}
__device__ __forceinline__ void v3_acc(vec4<float>& acc, const vec4<float>& A, const vec4<float>& B, const float* kA,
                                       const float* kB) {
  float2 a[4], b[4];
  float kab[4], k1[4], k2[4];
#pragma unroll
  for (int i = 0; i < 4; i++) {
    a[i] = pk(A.c[i]); b[i] = pk(B.c[i]);
    kab[i] = kA[i] - kB[i];
    k1[i] = kA[i] + 2.f * kB[i];
    k2[i] = -(2.f * kA[i] + kB[i]);
  }
  const float2 ab = mdot2(a, b), ca = mdot2(k1, a), cb = mdot2(k2, b);
#pragma unroll
  for (int i = 0; i < 4; i++) {
    float2 t = rmac2(pk(acc.c[i]), kab[i], ab);
    t = cmac2(t, ca, b[i]);
    t = cmac2(t, cb, a[i]);
    acc.c[i].re = t.x; acc.c[i].im = t.y;
  }
}
__device__ __forceinline__ void v4_acc(vec4<float>& acc, const vec4<float>& A, const vec4<float>& B, const vec4<float>& C) {
  float2 a[4], b[4], c[4];
#pragma unroll
  for (int i = 0; i < 4; i++) { a[i] = pk(A.c[i]); b[i] = pk(B.c[i]); c[i] = pk(C.c[i]); }
  float2 ac = mdot2(a, c);
  ac = __fadd2_rn(ac, ac);
  const float2 bc = mdot2(b, c), ab = mdot2(a, b);
#pragma unroll
  for (int i = 0; i < 4; i++) {
    float2 t = cmac2(pk(acc.c[i]), ac, b[i]);
    t = cmsc2(t, bc, a[i]);
    t = cmsc2(t, ab, c[i]);
    acc.c[i].re = t.x; acc.c[i].im = t.y;
  }
}

template <class G, typename T>
struct GrpGeom {
  // NGRP combinations per event, processed NPASS groups at a time (n = 4: all 16 at once; n = 5: shared memory
  // holds 12 of the 32)
  // HTL: both t helicities are walked by the same lane (every current loaded from shared memory feeds two
  // quark-line products); otherwise lanes are (s1, h_t) pairs
#ifdef ME_HTL
  static constexpr bool HTL = (ME_HTL != 0);
#else
  static constexpr bool HTL = (G::n <= 4);
#endif
  static constexpr int N = G::n, NHT = HTL ? 2 : 1, LPG = HTL ? N : 2 * N, GPW = 32 / LPG, NGRP = 1 << N;
  static constexpr int NPASS = (N <= 4) ? NGRP : 12;
  static constexpr int NW = (NPASS + GPW - 1) / GPW, NT = NW * 32;
  // T units per group: current slots + J[ncol][4][2]; padded so that the byte stride is 32 mod 128
  static constexpr int RAW = (G::nslot + G::ncol) * 8;
  static constexpr int UNIT = 32 / (int)sizeof(T);  // T units in 32 bytes
  static constexpr int GS = ((RAW + 4 * UNIT - 1) / (4 * UNIT)) * (4 * UNIT) + UNIT;
};

// Colour-ordered gluon currents of one group, level by level (|seq| = 2 .. n).  One copy of the vertex code: the
// levels, the tasks of a level and the terms of a task are run-time loops over the generated tables (keeps the
// kernel small enough for the instruction cache; the loop bodies are ~100 FMA-pipe instructions each).
template <class G, typename T, typename TC>
__device__ __forceinline__ void grp_tree(const GrpEvent<T, TC, G::n>& ev, T* slots, T* J, int r, bool active) {
  constexpr int LPG = GrpGeom<G, T>::LPG;
#pragma unroll 1
  for (int L = 2; L <= G::n; L++) {
    const int NV3 = L - 1, NV4 = (L - 1) * (L - 2) / 2, W = 2 + NV3 + NV4;
    const bool TOP = (L == G::n);
    const unsigned* tab = G::level(L);
    const int nt = G::ntask(L);
#pragma unroll 1
    for (int t0 = 0; t0 < nt; t0 += LPG) {
      const int t = t0 + r;
      if (active && t < nt) {
        const unsigned* tw = tab + t * W;
        const unsigned h0 = __ldg(tw);
        vec4<T> acc = zero_vec4<T>();
#pragma unroll 1
        for (int j = 0; j < NV3; j++) {
          const unsigned w = __ldg(tw + 2 + j);
          const vec4<T> A = GrpSlot<T>::ld(slots, w & 255u, w >> 31);
          const vec4<T> B = GrpSlot<T>::ld(slots, (w >> 8) & 255u, 0u);
          v3_acc(acc, A, B, ev.Ksub[(w >> 16) & 31u], ev.Ksub[(w >> 21) & 31u]);
        }
#pragma unroll 1
        for (int j = 0; j < NV4; j++) {
          const unsigned w = __ldg(tw + 2 + NV3 + j);
          const vec4<T> A = GrpSlot<T>::ld(slots, w & 255u, w >> 31);
          const vec4<T> B = GrpSlot<T>::ld(slots, (w >> 8) & 255u, 0u);
          const vec4<T> C = GrpSlot<T>::ld(slots, (w >> 16) & 255u, 0u);
          v4_acc(acc, A, B, C);
        }
        const T s = ev.ik[(h0 >> 8) & 31u];
#pragma unroll
        for (int i = 0; i < 4; i++) acc.c[i] = s * acc.c[i];
        if (!TOP) {
          GrpSlot<T>::st(slots, h0 & 255u, acc);
        } else {
          // the full-length current is contracted at once with the four t-tbar currents: initial J of the flow
          // and of its reverse
          const unsigned h1 = __ldg(tw + 1);
          T* ja = J + (h1 & 127u) * 8;
          T* jb = J + ((h1 >> 8) & 127u) * 8;
          const T sb = (h1 >> 31) ? T(-1) : T(1);
#pragma unroll
          for (int v = 0; v < 4; v++) {
            const vec4<T> q = GrpVec<T>::ld(ev.Q[v], 0u);
            const cx<T> a = mdot(q, acc);
            ja[2 * v] = a.re; ja[2 * v + 1] = a.im;
            jb[2 * v] = sb * a.re; jb[2 * v + 1] = sb * a.im;
          }
        }
      }
    }
    __syncwarp();
  }
}

// Quark-line walk of lane (s1, h_t): depth-first loop nest over the gluons that follow s1.  The words are read
// in execution order from the role's stream (emit_group.py role_stream); psi[j] = Psi(path[:j]) stays in registers.
template <class G, typename T, typename TC>
struct GrpWalkCtx {
  const GrpEvent<T, TC, G::n>* ev;
  const T* slots;
  T* J;
  const unsigned* stream;
  int ht;
  __device__ __forceinline__ unsigned next() { return __ldg(stream++); }
  __device__ __forceinline__ vec4<T> cur(unsigned w) const { return GrpSlot<T>::ld(slots, w & 255u, w >> 31); }
  typedef WalkPack<T, GrpGeom<G, T>::HTL> WP;
  typedef typename WP::PS PS;
  __device__ __forceinline__ vec4<PS> curw(unsigned w) const {
    const vec4<T> x = cur(w);
    vec4<PS> r;
#pragma unroll
    for (int i = 0; i < 4; i++) r.c[i] = mk<PS>(WP::widen(x.c[i].re), WP::widen(x.c[i].im));
    return r;
  }
  // external spinor(s) ubar(t) of chain c
  __device__ __forceinline__ spin4<PS> psi0(int c) const {
    spin4<PS> r;
    if constexpr (WP::NCH == 1 && GrpGeom<G, T>::HTL) {  // packed pair: (h_t = 0, h_t = 1)
      const spin4<T> a = ld_spin<T>(ev->ub[0]), b = ld_spin<T>(ev->ub[1]);
#pragma unroll
      for (int i = 0; i < 4; i++) r.c[i] = mk<PS>(pack(a.c[i].re, b.c[i].re), pack(a.c[i].im, b.c[i].im));
    } else {
      const spin4<T> a = ld_spin<T>(ev->ub[GrpGeom<G, T>::HTL ? c : ht]);
#pragma unroll
      for (int i = 0; i < 4; i++) r.c[i] = mk<PS>(WP::widen(a.c[i].re), WP::widen(a.c[i].im));
    }
    return r;
  }
  __device__ __forceinline__ static f2 pack(float x, float y) { return mkf2(x, y); }
  __device__ __forceinline__ static double pack(double x, double) { return x; }
  // Psi = X (qslash + m) / (q^2 - m^2 + i m Gamma) after the gluons of word w; q, the denominator and m are shared
  __device__ __forceinline__ static void addto(T* j, int h, int b, f2 re, f2 im) {
    j[0 * 4 + 2 * b] += re.v.x; j[0 * 4 + 2 * b + 1] += im.v.x;
    j[1 * 4 + 2 * b] += re.v.y; j[1 * 4 + 2 * b + 1] += im.v.y;
  }
  template <typename S> __device__ __forceinline__ static void addto(T* j, int h, int b, S re, S im) {
    j[h * 4 + 2 * b] += re; j[h * 4 + 2 * b + 1] += im;
  }
  __device__ __forceinline__ void leaf(const spin4<PS> (&X)[WP::NCH], unsigned w) const {
    T* j = J + ((w >> 16) & 127u) * 8;
#pragma unroll
    for (int b = 0; b < 2; b++) {
      const spin4<T> vb = ld_spin<T>(ev->v[b]);
      spin4<PS> vw;
#pragma unroll
      for (int i = 0; i < 4; i++) vw.c[i] = mk<PS>(WP::widen(vb.c[i].re), WP::widen(vb.c[i].im));
#pragma unroll
      for (int c = 0; c < WP::NCH; c++) {
        const cx<PS> a = row_col(X[c], vw);
        addto(j, GrpGeom<G, T>::HTL ? c : ht, b, a.re, a.im);
      }
    }
  }
};

// node whose path holds D gluons; psi[c][0..D-1] are valid on entry (c runs over the register chains of the lane)
template <class G, typename T, typename TC, int D>
struct GrpWalk {
  typedef GrpWalkCtx<G, T, TC> Ctx;
  typedef typename Ctx::PS PS;
  static constexpr int NCH = Ctx::WP::NCH;
  __device__ __forceinline__ static void node(Ctx& c, spin4<PS> (&psi)[NCH][G::n]) {
    const unsigned w0 = c.next();
    spin4<PS> X[NCH];
    {
      const vec4<PS> J0 = c.curw(w0);
#pragma unroll
      for (int h = 0; h < NCH; h++) X[h] = row_slash(psi[h][0], J0);
    }
#pragma unroll
    for (int j = 1; j < D; j++) {
      const vec4<PS> Jj = c.curw(c.next());
#pragma unroll
      for (int h = 0; h < NCH; h++) row_slash_add(X[h], psi[h][j], Jj);
    }
    {
      const unsigned m = (w0 >> 8) & 31u;
      mom4<PS> q;
#pragma unroll
      for (int i = 0; i < 4; i++) q.c[i] = Ctx::WP::widen(c.ev->qsub[m][i]);
      const cx<PS> gd = mk<PS>(Ctx::WP::widen(c.ev->gd[m][0]), Ctx::WP::widen(c.ev->gd[m][1]));
      const PS mt = Ctx::WP::widen(c.ev->mt);
#pragma unroll
      for (int h = 0; h < NCH; h++) psi[h][D] = row_prop(X[h], q, mt, gd);
    }
#pragma unroll 1
    for (int child = 0; child < G::n - D; child++) GrpWalk<G, T, TC, D + 1>::node(c, psi);
  }
};
template <class G, typename T, typename TC>
struct GrpWalk<G, T, TC, G::n> {
  typedef GrpWalkCtx<G, T, TC> Ctx;
  typedef typename Ctx::PS PS;
  static constexpr int NCH = Ctx::WP::NCH;
  __device__ __forceinline__ static void node(Ctx& c, spin4<PS> (&psi)[NCH][G::n]) {
    spin4<PS> X[NCH];
    {
      const vec4<PS> J1 = c.curw(c.next());
#pragma unroll
      for (int h = 0; h < NCH; h++) X[h] = row_slash(psi[h][1], J1);
    }
#pragma unroll
    for (int j = 2; j < G::n; j++) {
      const vec4<PS> Jj = c.curw(c.next());
#pragma unroll
      for (int h = 0; h < NCH; h++) row_slash_add(X[h], psi[h][j], Jj);
    }
    c.leaf(X, c.next());
  }
};

// x^T C x for the real vector x_a = J[a*8 + off] (a < ncol), C = integer numerators CM::at (symmetric)
template <int NCOL, typename T, typename TC, class CM>
__device__ __forceinline__ TC grp_quadform(const T* J, int off, TC* x2 /*[NCOL] += x_a^2 or nullptr*/, TC keep) {
  static_assert(NCOL <= 24, "register-resident form (120 flows: the row-split loop of the kernel)");
  TC s = TC(0);
  {
    TC x[NCOL];
#pragma unroll
    for (int a = 0; a < NCOL; a++) x[a] = TC(J[a * 8 + off]);
#pragma unroll
    for (int a = 0; a < NCOL; a++) {
      TC y = TC(0.5) * CM::at(a * NCOL + a) * x[a];
#pragma unroll
      for (int b = a + 1; b < NCOL; b++) y += CM::at(a * NCOL + b) * x[b];
      s += x[a] * y;
      if (x2) x2[a] += keep * x[a] * x[a];
    }
  }
  return TC(2) * s;
}

// One warp: in-order cumulative sums of PER consecutive values per lane (index = lane * PER + i; val = 0 where
// !ok), their total, and the selection of reading R11: first index with rnd * total < cumulative sum, else the last
// ok index.  Every lane returns the same total and sel.
template <int PER>
__device__ __forceinline__ void grp_warp_select(const double (&val)[PER], const bool (&ok)[PER], double rnd, int lane,
                                                double& total, int& sel) {
  double pre[PER], run = 0.0;
#pragma unroll
  for (int i = 0; i < PER; i++) { run += val[i]; pre[i] = run; }
  double inc = run;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const double t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  const double off = inc - run;
  total = __shfl_sync(0xffffffffu, inc, 31);
  const double target = rnd * total;
  int hit = -1, lastok = -1;
#pragma unroll
  for (int i = 0; i < PER; i++) {
    if (hit < 0 && ok[i] && target < off + pre[i]) hit = lane * PER + i;
    if (ok[i]) lastok = lane * PER + i;
  }
  const unsigned bh = __ballot_sync(0xffffffffu, hit >= 0), bo = __ballot_sync(0xffffffffu, lastok >= 0);
  if (bh) sel = __shfl_sync(0xffffffffu, hit, __ffs(bh) - 1);
  else sel = bo ? __shfl_sync(0xffffffffu, lastok, 31 - __clz(bo)) : 0;
}

// float colour sum of one variant (h_t, h_tbar) with the real and imaginary parts of J as one packed f32x2 pair
// (inline PTX on 64-bit registers: arrays of them unroll like scalars, arrays of float2 through the builtins did
// not): returns Re(J^dagger C J) = x^T C x + y^T C y for J = x + i y, J_a at J[a*8 + 2*v .. +1]
__device__ __forceinline__ unsigned long long pk2(float x, float y) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
  return r;
}
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
  unsigned long long r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ unsigned long long mul2(unsigned long long a, unsigned long long b) {
  unsigned long long r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
template <int NCOL, typename T, class CM>
__device__ __forceinline__ float grp_quadform_pk(const T* J, int v, float* x2 /*[NCOL] += |J_a|^2 or nullptr*/, float keep) {
  static_assert(NCOL <= 24, "register-resident form");
  unsigned long long x[NCOL];
  float xr[NCOL], xi[NCOL];
#pragma unroll
  for (int a = 0; a < NCOL; a++) {
    xr[a] = float(J[a * 8 + 2 * v]); xi[a] = float(J[a * 8 + 2 * v + 1]);
    x[a] = pk2(xr[a], xi[a]);
  }
  unsigned long long s = pk2(0.f, 0.f);
#pragma unroll
  for (int a = 0; a < NCOL; a++) {
    const float caa = 0.5f * CM::at(a * NCOL + a);
    unsigned long long y = mul2(pk2(caa, caa), x[a]);
#pragma unroll
    for (int b = a + 1; b < NCOL; b++) {
      const float c = CM::at(a * NCOL + b);
      y = fma2(pk2(c, c), x[b], y);
    }
    s = fma2(x[a], y, s);
    if (x2) x2[a] += keep * (xr[a] * xr[a] + xi[a] * xi[a]);
  }
  float sx, sy;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(sx), "=f"(sy) : "l"(s));
  return 2.f * (sx + sy);
}
template <typename TC> struct GrpIsFloat { static constexpr bool value = false; };
template <> struct GrpIsFloat<float> { static constexpr bool value = true; };

template <class G, typename T, typename TC, class CM, int MODE, int MINB>
__global__ void __launch_bounds__(GrpGeom<G, T>::NT, MINB) group_kernel(const LaunchArgs a) {
  typedef GrpGeom<G, T> GE;
  constexpr int N = G::n, NPAR = N + 2, NCOMB = 1 << NPAR, LPG = GE::LPG, GPW = GE::GPW, NT = GE::NT;
  typedef GrpEvent<T, TC, N> EV;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  EV& ev = *reinterpret_cast<EV*>(smem_raw);
  T* gbase = reinterpret_cast<T*>(smem_raw + ((sizeof(EV) + 127) / 128) * 128);
  // optional shared-memory copy of the colour matrix as 16-bit integers (behind the group areas), made once
  const short* cm16 = reinterpret_cast<const short*>(gbase + (size_t)GrpGeom<G, T>::NPASS * GrpGeom<G, T>::GS);
  if constexpr (CM::smem16) {
    const int4* src = reinterpret_cast<const int4*>(CM::table16());
    int4* dst = reinterpret_cast<int4*>(const_cast<short*>(cm16));
    for (int i = threadIdx.x; i < (G::ncol * G::ncol * 2 + 15) / 16; i += GrpGeom<G, T>::NT) dst[i] = __ldg(src + i);
  }
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int gi = lane / LPG, r = lane - gi * LPG;
  const int lgrp = warp * GPW + gi;                      // group slot of this lane within a pass
  T* slots = gbase + (size_t)((gi < GPW && lgrp < GE::NPASS) ? lgrp : 0) * GE::GS;
  T* J = slots + G::nslot * 8;
  const double mw = a.par.mt * a.par.wt;

  for (long long e = blockIdx.x; e < a.nevt; e += gridDim.x) {
    __syncthreads();
    // ---- a1 + per-event, helicity-independent data (a2 bases, invariants in fp64) in ONE phase: every task reads
    // the momenta it needs from global memory (L1-resident after the first touch; incoming convention: +p for the
    // initial, -p for the final state), so no task waits for another and one block barrier ends the setup
    const double* pm = a.mom + e * (NPAR * 4);
    auto kd = [&](int p, int c) { const double x = __ldg(pm + 4 * p + c); return (p < 2) ? x : -x; };
    auto dot2 = [&](int p, int q) {  // 2 k_p . k_q
      return 2.0 * (kd(p, 0) * kd(q, 0) - kd(p, 1) * kd(q, 1) - kd(p, 2) * kd(q, 2) - kd(p, 3) * kd(q, 3));
    };
    if (tid == 0) ev.mt = T(a.par.mt);
    auto is_good = [&](int h) { return MODE == MODE_FILTER || ((a.good.mask[h >> 6] >> (h & 63)) & 1ull) != 0ull; };
    auto hel_of = [&](int gg, int v) {  // helicity row of gluon-helicity combination gg and variant v = 2 h_t + h_tbar
      int h = 0;
      for (int i = 0; i < N; i++) {
        const int p = (i < 2) ? i : i + 2;
        h |= ((gg >> (N - 1 - i)) & 1) << (NPAR - 1 - p);
      }
      h |= (v >> 1) << (NPAR - 1 - 2);
      h |= (v & 1) << (NPAR - 1 - 3);
      return h;
    };
    if (MODE == MODE_SELECT && tid >= NT - GE::NGRP) {  // the last NGRP threads: good-helicity bits per combination
      const int gg = tid - (NT - GE::NGRP);
      int m = 0;
      for (int v = 0; v < 4; v++) m |= is_good(hel_of(gg, v)) ? (1 << v) : 0;
      ev.gmask[gg] = (unsigned char)m;
    }
    // the subset tasks run on warp 0, the wavefunction tasks on warp 1: different task types in one warp would
    // diverge and run one after the other, and this section is pure latency for the whole block
    static_assert((1 << N) <= 32 && NT >= 32 + N + 6, "setup task layout");
    {
      const int task = (tid < (1 << N)) ? tid : ((tid >= 32 && tid < 32 + N + 6) ? (1 << N) + tid - 32 : -1);
      if (task < 0) {
      } else if (task < (1 << N)) {
        // gluon subset m: momentum sum, quark-line momentum after it, 1/K^2, quark-line denominator.
        // Branch-free: every lane loads all gluon momenta and forms every 2 k_i.k_j, members are picked with
        // 0/1 factors (exact), so the latency of this serial section is one round of loads + ~150 FP64 operations
        const int m = task;
        double kg[N][4], kt[4];
#pragma unroll
        for (int i = 0; i < N; i++)
#pragma unroll
          for (int c = 0; c < 4; c++) kg[i][c] = kd((i < 2) ? i : i + 2, c);
#pragma unroll
        for (int c = 0; c < 4; c++) kt[c] = kd(2, c);
        double k[4] = {0.0, 0.0, 0.0, 0.0}, pairs = 0.0, line = 0.0;
#pragma unroll
        for (int i = 0; i < N; i++) {
          const double bi = ((m >> i) & 1) ? 1.0 : 0.0;
#pragma unroll
          for (int c = 0; c < 4; c++) k[c] += bi * kg[i][c];
          line += bi * 2.0 * (kt[0] * kg[i][0] - kt[1] * kg[i][1] - kt[2] * kg[i][2] - kt[3] * kg[i][3]);
#pragma unroll
          for (int j = i + 1; j < N; j++) {
            const double bj = ((m >> j) & 1) ? bi : 0.0;
            pairs += bj * 2.0 * (kg[i][0] * kg[j][0] - kg[i][1] * kg[j][1] - kg[i][2] * kg[j][2] - kg[i][3] * kg[j][3]);
          }
        }
        const int cnt = __popc(m);
        for (int c = 0; c < 4; c++) {
          ev.Ksub[m][c] = T(k[c]);
          ev.qsub[m][c] = T(-(kt[c] + k[c]));
        }
        ev.ik[m] = (cnt >= 2) ? T(1.0 / pairs) : T(0);
        const double den = line + pairs, nrm = 1.0 / (den * den + mw * mw);
        ev.gd[m][0] = (cnt >= 1) ? T(den * nrm) : T(0);
        ev.gd[m][1] = (cnt >= 1) ? T(-mw * nrm) : T(0);
      } else if (task < (1 << N) + N) {
        const int i = task - (1 << N), p = (i < 2) ? i : i + 2;
        mom4<T> k;
        for (int c = 0; c < 4; c++) k.c[c] = T(kd(p, c));
        const polbasis<T> pb = make_polbasis<T>((p < 2) ? k : neg(k));
        for (int c = 0; c < 3; c++) { ev.pol[i][c] = pb.e1[c]; ev.pol[i][3 + c] = pb.e2[c]; }
      } else {
        // tasks 0,1: ubar(t), v(tbar) for both helicities; tasks 2..5: Q(h_t, h_tbar) = ubar gamma^mu v
        const int w = task - (1 << N) - N;
        spin4<T> ub[2], vv[2];
#pragma unroll
        for (int which = 0; which < 2; which++) {
          mom4<T> k;
#pragma unroll
          for (int c = 0; c < 4; c++) k.c[c] = T(-kd(2 + which, c));
          const spinbasis<T> sb = make_spinbasis<T>(k, T(a.par.mt));
#pragma unroll
          for (int l = 0; l < 2; l++) {
            if (which) vv[l] = spinor_v(sb, l ? 1 : -1);
            else ub[l] = bar(spinor_u(sb, l ? 1 : -1));
          }
        }
        if (w < 2) {
#pragma unroll
          for (int l = 0; l < 2; l++) {
            T* o = w ? ev.v[l] : ev.ub[l];
#pragma unroll
            for (int c = 0; c < 4; c++) {
              o[2 * c] = w ? vv[l].c[c].re : ub[l].c[c].re;
              o[2 * c + 1] = w ? vv[l].c[c].im : ub[l].c[c].im;
            }
          }
        } else {
          const int v = w - 2;
          vec4<T> JR, JL;
          chiral_currents(select((v >> 1) != 0, ub[1], ub[0]), select((v & 1) != 0, vv[1], vv[0]), JR, JL);
          for (int c = 0; c < 4; c++) { ev.Q[v][2 * c] = JR.c[c].re + JL.c[c].re; ev.Q[v][2 * c + 1] = JR.c[c].im + JL.c[c].im; }
        }
      }
    }
    __syncthreads();
    if (MODE == MODE_SELECT)  // colour weights of this warp's groups (a8), accumulated over the passes
      for (int c = lane; c < G::ncol; c += 32) ev.wc[warp][c] = TC(0);
#pragma unroll 1
    for (int pass0 = 0; pass0 < GE::NGRP; pass0 += GE::NPASS) {
    const int grp = pass0 + lgrp;                        // gluon-helicity combination
    const bool active = (gi < GPW) && (lgrp < GE::NPASS) && (grp < GE::NGRP);
    // ---- a2: polarisation vectors of this group's gluon helicities
    if (active && r < N) {
      const int p = (r < 2) ? r : r + 2;
      const int lam = ((grp >> (N - 1 - r)) & 1) ? 1 : -1;
      polbasis<T> pb;
      for (int c = 0; c < 3; c++) { pb.e1[c] = ev.pol[r][c]; pb.e2[c] = ev.pol[r][3 + c]; }
      GrpSlot<T>::st(slots, r, polvec(pb, lam, p >= 2));
    }
    __syncwarp();
    // ---- a3: colour-ordered gluon currents, level by level; the full-length ones initialise J
    grp_tree<G, T, TC>(ev, slots, J, r, active);
    // ---- a3-a5: quark line
    if (active) {
      GrpWalkCtx<G, T, TC> c;
      c.ev = &ev; c.slots = slots; c.J = J;
      c.stream = G::role(GE::HTL ? r : (r >> 1));
      c.ht = GE::HTL ? 0 : (r & 1);
      typedef GrpWalkCtx<G, T, TC> Ctx;
      spin4<typename Ctx::PS> psi[Ctx::WP::NCH][G::n];
#pragma unroll
      for (int h = 0; h < Ctx::WP::NCH; h++) psi[h][0] = c.psi0(h);
      GrpWalk<G, T, TC, 1>::node(c, psi);
    }
    __syncwarp();
    // ---- a6: colour sums.  Helicity row of variant v = 2 h_t + h_tbar of this group:
    auto hel_row = [&](int v) { return hel_of(grp, v); };
    if constexpr (G::ncol > 24) {
      // rows of C split over the lanes of the group; every C_ab read once feeds the 8 real vectors
      // (4 variants x re/im) of the group; partial sums meet in the (now free) current slots
      TC part[8];
#pragma unroll
      for (int k = 0; k < 8; k++) part[k] = TC(0);
      if (active) {
        // RB rows of the lane at a time: every x_b fetched from shared memory feeds RB rows (the loop is bound by
        // shared-memory wavefronts: the lanes are at different b, nothing is broadcast)
        constexpr int RB = 4;
        auto cmat = [&](int i) { return CM::smem16 ? TC(cm16[i]) : CM::at(i); };
#pragma unroll 1
        for (int a0 = r; a0 < G::ncol; a0 += RB * LPG) {
          TC xa[RB][8], y[RB][8];
          int row[RB];
#pragma unroll
          for (int j = 0; j < RB; j++) {
            const int aj = a0 + j * LPG;
            const bool on = aj < G::ncol;
            row[j] = on ? aj : G::ncol - 1;
            const vec4<T> ja = GrpVec<T>::ld(J + row[j] * 8, 0u);
#pragma unroll
            for (int k = 0; k < 4; k++) { xa[j][2 * k] = on ? TC(ja.c[k].re) : TC(0); xa[j][2 * k + 1] = on ? TC(ja.c[k].im) : TC(0); }
            const TC caa = TC(0.5) * cmat(row[j] * G::ncol + row[j]);
#pragma unroll
            for (int k = 0; k < 8; k++) y[j][k] = caa * xa[j][k];
            if (!on) row[j] = G::ncol;  // no column b > row: contributes nothing
          }
#pragma unroll 2
          for (int b = a0 + 1; b < G::ncol; b++) {
            const vec4<T> jb = GrpVec<T>::ld(J + b * 8, 0u);
#pragma unroll
            for (int j = 0; j < RB; j++) {
              const TC c = (b > row[j]) ? cmat(row[j] * G::ncol + b) : TC(0);
#pragma unroll
              for (int k = 0; k < 4; k++) { y[j][2 * k] += c * TC(jb.c[k].re); y[j][2 * k + 1] += c * TC(jb.c[k].im); }
            }
          }
#pragma unroll
          for (int j = 0; j < RB; j++)
#pragma unroll
            for (int k = 0; k < 8; k++) part[k] += xa[j][k] * y[j][k];
        }
      }
      __syncwarp();  // every lane of the group is done with the current slots
      if (active) {
        vec4<T> pv;
#pragma unroll
        for (int k = 0; k < 4; k++) pv.c[k] = mk<T>(T(part[2 * k]), T(part[2 * k + 1]));
        GrpVec<T>::st(slots + r * 8, pv);
      }
      __syncwarp();
      if (active && r < 4) {
        double q = 0.0;
        for (int l = 0; l < LPG; l++) q += (double)slots[l * 8 + 2 * r] + (double)slots[l * 8 + 2 * r + 1];
        ev.mh[hel_row(r)] = 2.0 * q;
      }
    } else if constexpr (GrpIsFloat<TC>::value) {
      // float colour sum: task = variant (4 per group), re and im of J as one packed f32x2 pair
#pragma unroll 1
      for (int k0 = 0; k0 < 4; k0 += LPG) {
        const int v = k0 + r;
        if (active && v < 4) {
          const int h = hel_row(v);
          const float keep = is_good(h) ? 1.f : 0.f;
          ev.mh[h] = (double)grp_quadform_pk<G::ncol, T, CM>(J, v, nullptr, keep);
        }
      }
    } else {
      // task = (variant, re/im): 8 per group, lane r takes tasks r, r + LPG, ...; pairs are added by one shuffle
#pragma unroll 1
      for (int k0 = 0; k0 < 8; k0 += LPG) {
        const int k = k0 + r;
        TC q = TC(0);
        int h = 0;
        const bool on = active && k < 8;
        if (on) {
          h = hel_row(k >> 1);
          const TC keep = is_good(h) ? TC(1) : TC(0);
          q = grp_quadform<G::ncol, T, TC, CM>(J, k, nullptr, keep);
        }
        q += __shfl_xor_sync(0xffffffffu, q, 1);
        if (on && !(k & 1)) ev.mh[h] = (double)q;
      }
    }
    __syncwarp();
    if (MODE == MODE_SELECT) {
      // a8 colour weights w_c += sum over this warp's groups and the good (h_t, h_tbar) of |J_c|^2: lane = flow,
      // read back from the J areas (cheaper than per-lane partial sums and a shuffle reduction per flow)
      for (int c = lane; c < G::ncol; c += 32) {
        TC w = TC(0);
#pragma unroll 1
        for (int g = 0; g < GPW; g++) {
          const int lg = warp * GPW + g, gg = pass0 + lg;
          if (lg < GE::NPASS && gg < GE::NGRP) {
            const vec4<T> j = GrpVec<T>::ld(gbase + (size_t)lg * GE::GS + G::nslot * 8 + c * 8, 0u);
            const int gm = ev.gmask[gg];
#pragma unroll
            for (int v = 0; v < 4; v++) {
              const TC keep = ((gm >> v) & 1) ? TC(1) : TC(0);
              w += keep * (TC(j.c[v].re) * TC(j.c[v].re) + TC(j.c[v].im) * TC(j.c[v].im));
            }
          }
        }
        ev.wc[warp][c] += w;
      }
      __syncwarp();
    }
    }  // passes
    __syncthreads();
    // ---- a7-a9
    if (MODE == MODE_FILTER) {
      double total = 0.0;
      for (int h = 0; h < NCOMB; h++) total += ev.mh[h];
      for (int h = tid; h < NCOMB; h += NT) {
        const double f = (total > 0.0) ? ev.mh[h] / total : 0.0;
        atomicMax(a.fracmax + h, (unsigned long long)__double_as_longlong(f));
      }
    } else if (warp == 0) {
      // helicity sum in table order (a7), ME (a9) and helicity selection (a8): one warp, in-order scan
      constexpr int PER = NCOMB / 32;
      double val[PER];
      bool ok[PER];
#pragma unroll
      for (int i = 0; i < PER; i++) {
        const int h = lane * PER + i;
        ok[i] = is_good(h);
        val[i] = ok[i] ? ev.mh[h] : 0.0;
      }
      double total;
      int sel;
      grp_warp_select<PER>(val, ok, (MODE == MODE_SELECT && a.selhel) ? a.rndhel[e] : 0.0, lane, total, sel);
      if (lane == 0) {
        const double g = a.gs[e];
        a.me[e] = total * ipow<2 * N>(g) * (1.0 / (double(G::denom) * double(G::cden)));
        if (MODE == MODE_SELECT && a.selhel) a.selhel[e] = sel;
      }
    } else if (warp == 1 && MODE == MODE_SELECT && a.selcol) {
      constexpr int PER = (G::ncol + 31) / 32;
      double val[PER];
      bool ok[PER];
#pragma unroll
      for (int i = 0; i < PER; i++) {
        const int c = lane * PER + i;
        ok[i] = c < G::ncol;
        TC w = TC(0);
        if (ok[i])
          for (int k = 0; k < GE::NW; k++) w += ev.wc[k][c];
        val[i] = (double)w;
      }
      double total;
      int sel;
      grp_warp_select<PER>(val, ok, a.rndcol[e], lane, total, sel);
      if (lane == 0) a.selcol[e] = sel;
    }
  }
}

}  // namespace me
