// me_group.cuh -- the "lane-group" pipeline (layout B2) for g g -> t tbar + (n-2) g, n >= 4: three kernels per chunk
// of events, the amplitudes on the FMA pipes and the colour contraction on the tensor cores.
//
//   K0 setup_kernel   a1 + the helicity-independent part of a2/a3: momentum sums per gluon subset,
//                     1/K^2, quark-line denominators (formed in fp64 from pairwise invariants, whatever the build),
//                     polarisation / spinor bases, the four t-tbar currents Q(h_t,h_tbar) -> GrpEvent[event] in HBM.
//   K1 amp_kernel     a2-a5.  One WARP per (event, unit); a GROUP of LPG lanes owns one combination of the n gluon
//                     helicities (n = 4: 4 lanes, one per first gluon s1 of the colour flow, both t helicities walked
//                     by the same lane; n = 5: 10 lanes (s1, h_t)), so the gluon currents are computed once per
//                     gluon-helicity combination and shared by the four (h_t, h_tbar) rows.  Warp-synchronous:
//                       leaves  lane i < n      : polarisation vector of gluon i                    -> shared-memory slot
//                       tree    lane = sequence : colour-ordered currents Jord(seq), |seq| = 2..n-1 -> shared-memory slot
//                               |seq| = n       : contracted at once with the four Q               -> "init" slot
//                       walk    lane = s1       : quark line for the flows that start with gluon s1; at the leaf of
//                               flow sigma  J_sigma = init + Psi.v  goes straight to HBM as X[event][combination][flow][8]
//                               (8 = 2 (2 h_t + h_tbar) + re/im; 16- or 32-byte stores): the jamps never sit in
//                               shared memory.
//   K2 colour_kernel  a6-a9.  One warp per event.  Per gluon-helicity combination the colour sum of its 8 real
//                     vectors is the contraction  q_m = sum_ab X[m][a] C[a][b] X[m][b]  = [8 x ncol] . [ncol x ncol]
//                     followed by a row dot: tensor-core MMAs with X loaded from HBM straight into A fragments
//                     (256 / 128 contiguous bytes per warp load), C in shared memory in fragment order, only the
//                     upper triangle of 8 x 8 tiles (diagonal tiles halved, result doubled: C is symmetric); the
//                     columns of every tile are permuted so that the D fragment of a thread meets the X values it
//                     already holds (the row dot needs no second load).
//                       fp64 build        : mma.sync m8n8k4 f64 (DMMA)
//                       fp32 / mixed build: mma.sync m16n8k8 tf32, two combinations per tile, X split into
//                                           hi + lo TF32 parts (the integer colour numerators are exact in TF32), so
//                                           the products carry fp32 accuracy and the sum accumulates in fp32
//                     then |M_h|^2 per helicity row, the helicity sum in table order (a7), helicity / colour selection
//                     (a8) and the stores (a9).
// The fp32 build packs the two h_t chains of the walk, the complex arithmetic of the tree vertices into f32x2
// operations (FFMA2).  DESIGN.md section 5 has the measured history of these choices.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "me_kernels.cuh"

#ifndef ME_UNROLL_T
#define ME_UNROLL_T 1   // unroll factor of the term loops of the tree (loads of term j + 1 overlap the arithmetic of term j)
#endif

// -DME_CHECK=1: the build of the self-checks (compute-sanitizer is not available on the pool):
// every slot index read from a table is bounds-checked, the shared memory of a warp and the pipeline scratch of a
// chunk are filled with NaN before use, so that a read of anything not written in this unit / chunk shows up as a
// NaN matrix element in the parity tests
#if defined(ME_CHECK) && ME_CHECK
#include <cassert>
#define ME_ASSERT(x) assert(x)
#else
#define ME_ASSERT(x) ((void)0)
#endif

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
  template <bool SIGNS = true>
  __device__ __forceinline__ static vec4<double> ld(const double* slots, unsigned s, unsigned neg) {
    const char* base = reinterpret_cast<const char*>(slots + s * 8);
    const unsigned x = (s >> 1) & 3u;
    const int m = SIGNS ? (int)(neg << 31) : 0;
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
  template <bool SIGNS = true>
  __device__ __forceinline__ static vec4<float> ld(const float* slots, unsigned s, unsigned neg) {
    const char* base = reinterpret_cast<const char*>(slots + s * 8);
    const unsigned x = 0u;  // fp32: the extra address arithmetic costs more issue slots than the conflicts (measured)
    const int m = SIGNS ? (int)(neg << 31) : 0;
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

// a or -a (neg = 1): sign bits flipped on the integer pipe
__device__ __forceinline__ vec4<double> vsgn(const vec4<double>& a, unsigned neg) {
  const int m = (int)(neg << 31);
  vec4<double> r;
#pragma unroll
  for (int i = 0; i < 4; i++) {
    r.c[i].re = __hiloint2double(__double2hiint(a.c[i].re) ^ m, __double2loint(a.c[i].re));
    r.c[i].im = __hiloint2double(__double2hiint(a.c[i].im) ^ m, __double2loint(a.c[i].im));
  }
  return r;
}
__device__ __forceinline__ vec4<float> vsgn(const vec4<float>& a, unsigned neg) {
  const int m = (int)(neg << 31);
  vec4<float> r;
#pragma unroll
  for (int i = 0; i < 4; i++) {
    r.c[i].re = __int_as_float(__float_as_int(a.c[i].re) ^ m);
    r.c[i].im = __int_as_float(__float_as_int(a.c[i].im) ^ m);
  }
  return r;
}

// acc += (A.B)(kA-kB) + ((kA+2kB).A) B - ((2kA+kB).B) A      (three-gluon vertex, propagator applied later)
// kB is not loaded: with Kt = kA + kB the momentum of the task's sequence (one load per task, kt2 = 2 Kt),
// kA - kB = 2 kA - Kt,  kA + 2 kB = 2 Kt - kA,  -(2 kA + kB) = -(kA + Kt): the tree is bound by shared-memory traffic
template <typename T>
__device__ __forceinline__ void v3_acc(vec4<T>& acc, const vec4<T>& A, const vec4<T>& B, const T* kA, const T (&kt)[4], const T (&kt2)[4]) {
  const cx<T> ab = mdot(A, B);
  mom4<T> kab, k1, k2;
#pragma unroll
  for (int i = 0; i < 4; i++) {
    kab.c[i] = T(2) * kA[i] - kt[i];
    k1.c[i] = kt2[i] - kA[i];
    k2.c[i] = -(kA[i] + kt[i]);
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
                                       const float (&kt)[4], const float (&kt2)[4]) {
  float2 a[4], b[4];
  float kab[4], k1[4], k2[4];
#pragma unroll
  for (int i = 0; i < 4; i++) {
    a[i] = pk(A.c[i]); b[i] = pk(B.c[i]);
    kab[i] = 2.f * kA[i] - kt[i];
    k1[i] = kt2[i] - kA[i];
    k2[i] = -(kA[i] + kt[i]);
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


// Accumulator of one tree task.  fp64: the current itself.  fp32: the sum is kept as TWO packed accumulators per
// component, acc_i = P_i + i Q_i with P_i, Q_i complex pairs: a complex product c * v adds c.re * v to P and c.im * v
// to Q, i.e. two FFMA2 whose first operand is a broadcast scalar and whose second is the pair as loaded -- no
// swapped / sign-flipped copies of either factor (they cost 17 moves and 6 negations per three-gluon term in the
// single-accumulator form; measured).  P + i Q is folded once per task in finish().
template <typename T> struct TreeAcc {
  vec4<T> acc;
  __device__ __forceinline__ void zero() { acc = zero_vec4<T>(); }
  __device__ __forceinline__ void v3(const vec4<T>& A, const vec4<T>& B, const T* kA, const T (&kt)[4], const T (&kt2)[4]) { v3_acc(acc, A, B, kA, kt, kt2); }
  __device__ __forceinline__ void v4(const vec4<T>& A, const vec4<T>& B, const vec4<T>& C) { v4_acc(acc, A, B, C); }
  __device__ __forceinline__ vec4<T> finish(T s) const {
    vec4<T> r;
#pragma unroll
    for (int i = 0; i < 4; i++) r.c[i] = s * acc.c[i];
    return r;
  }
};
// Minkowski product of two complex vectors as (P, Q): a.b = P + i Q, P = sum g_i a_i.re b_i, Q = sum g_i a_i.im b_i
__device__ __forceinline__ float2 fold_pq(float2 P, float2 Q) { return make_float2(P.x - Q.y, P.y + Q.x); }
__device__ __forceinline__ float2 mdot_pq(const float2 (&A)[4], const float2 (&B)[4]) {
  float2 P = __fmul2_rn(make_float2(A[0].x, A[0].x), B[0]);
  float2 Q = __fmul2_rn(make_float2(A[0].y, A[0].y), B[0]);
#pragma unroll
  for (int i = 1; i < 4; i++) {
    P = __ffma2_rn(make_float2(-A[i].x, -A[i].x), B[i], P);
    Q = __ffma2_rn(make_float2(-A[i].y, -A[i].y), B[i], Q);
  }
  return fold_pq(P, Q);
}
template <> struct TreeAcc<float> {
  float2 P[4], Q[4];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int i = 0; i < 4; i++) P[i] = Q[i] = make_float2(0.f, 0.f);
  }
  // += c * v   /   -= c * v
  __device__ __forceinline__ void mac(int i, float2 c, float2 v) {
    P[i] = __ffma2_rn(make_float2(c.x, c.x), v, P[i]);
    Q[i] = __ffma2_rn(make_float2(c.y, c.y), v, Q[i]);
  }
  __device__ __forceinline__ void msc(int i, float2 c, float2 v) {
    P[i] = __ffma2_rn(make_float2(-c.x, -c.x), v, P[i]);
    Q[i] = __ffma2_rn(make_float2(-c.y, -c.y), v, Q[i]);
  }
  __device__ __forceinline__ void v3(const vec4<float>& A, const vec4<float>& B, const float* kA, const float (&kt)[4], const float (&kt2)[4]) {
    float2 a[4], b[4];
    float kab[4], k1[4], k2[4];
#pragma unroll
    for (int i = 0; i < 4; i++) {
      a[i] = pk(A.c[i]); b[i] = pk(B.c[i]);
      kab[i] = 2.f * kA[i] - kt[i];
      k1[i] = kt2[i] - kA[i];
      k2[i] = -(kA[i] + kt[i]);
    }
    const float2 ab = mdot_pq(a, b), ca = mdot2(k1, a), cb = mdot2(k2, b);
#pragma unroll
    for (int i = 0; i < 4; i++) {
      P[i] = rmac2(P[i], kab[i], ab);
      mac(i, ca, b[i]);
      mac(i, cb, a[i]);
    }
  }
  __device__ __forceinline__ void v4(const vec4<float>& A, const vec4<float>& B, const vec4<float>& C) {
    float2 a[4], b[4], c[4];
#pragma unroll
    for (int i = 0; i < 4; i++) { a[i] = pk(A.c[i]); b[i] = pk(B.c[i]); c[i] = pk(C.c[i]); }
    float2 ac = mdot_pq(a, c);
    ac = __fadd2_rn(ac, ac);
    const float2 bc = mdot_pq(b, c), ab = mdot_pq(a, b);
#pragma unroll
    for (int i = 0; i < 4; i++) {
      mac(i, ac, b[i]);
      msc(i, bc, a[i]);
      msc(i, ab, c[i]);
    }
  }
  __device__ __forceinline__ vec4<float> finish(float s) const {
    vec4<float> r;
#pragma unroll
    for (int i = 0; i < 4; i++) {
      const float2 t = __fmul2_rn(make_float2(s, s), fold_pq(P[i], Q[i]));
      r.c[i].re = t.x; r.c[i].im = t.y;
    }
    return r;
  }
};

// Helicity-independent data of one event: written by setup_kernel (K0) to HBM, staged in shared memory by the warp
// that evaluates a unit of the event (K1).
template <typename T, int N>
struct alignas(16) GrpEvent {
  alignas(16) T Ksub[1 << N][4];  // sum of the gluon momenta of a subset (bit i = gluon i)
  alignas(16) T qsub[1 << N][4];  // -(k_t + K_S): momentum of the quark line after the gluons of S
  T gd[1 << N][2];                // 1 / (q^2 - m^2 + i m Gamma)
  T ik[1 << N];                   // 1 / K_S^2
  alignas(16) T Q[4][8];          // ubar(h_t) gamma^mu v(h_tbar), index 2 h_t + h_tbar
  alignas(16) T ub[2][8];
  alignas(16) T v[2][8];
  T pol[N][6];
  T mt;
};

// Where the contracted full-length currents ("init": the j = 0 term of every jamp) wait for the walk: in the jamp
// buffer itself (HBM/L2; the leaf reads, adds and overwrites) when shared memory bounds the number of resident warps
// (n = 5: 6 -> 9 warps per SM in fp64, measured +9 % fp64, +30 % mixed), in shared memory when registers do (n = 4:
// the extra global round trip costs 7-15 %, measured).
template <class G> struct GrpInit {
#ifdef ME_INIT_GLOBAL
  static constexpr bool GLOBAL = (ME_INIT_GLOBAL != 0);
#else
  static constexpr bool GLOBAL = (G::n >= 5);
#endif
};

template <class G, typename T>
struct GrpGeom {
  // HTL: both t helicities are walked by the same lane (every current loaded from shared memory feeds two
  // quark-line products); otherwise lanes are (s1, h_t) pairs
#ifdef ME_HTL
  static constexpr bool HTL = (ME_HTL != 0);
#else
  static constexpr bool HTL = (G::n <= 4);
#endif
  static constexpr int N = G::n, NHT = HTL ? 2 : 1, LPG = HTL ? N : 2 * N, GPW = 32 / LPG, NGRP = 1 << N;
  // T units per group: current slots + contracted full-length currents ("init"); padded so that the byte stride
  // is 32 mod 128
  static constexpr int RAW = (G::nslot + (GrpInit<G>::GLOBAL ? 0 : G::ninit)) * 8;
  static constexpr int UNIT = 32 / (int)sizeof(T);  // T units in 32 bytes
  // Group stride = a multiple of 128 bytes + PAD.  The lanes r of neighbouring groups read the same slot numbers (same
  // tables), so the pad decides whether the two groups of a quarter-warp meet in the same banks: fp64 (64-byte slots,
  // chunk swizzle) 32 bytes; fp32 (32-byte slots at 2 (s mod 4) + chunk) 16 bytes, which puts the second group on the odd
  // 16-byte positions (modelled wavefronts of the slot accesses of gg_ttgg 588 -> 382 per group pair, ideal 192; measured
  // +4.8 % gg_ttgg fp32, +3.4 % gg_ttggg fp32; the fp64 builds are best at 32: pads 16 / 48 / 64 measured 2-4 % slower)
#ifdef ME_GS_PAD_BYTES
  static constexpr int PAD = ME_GS_PAD_BYTES / (int)sizeof(T);
#else
  static constexpr int PAD = (sizeof(T) == 4) ? 16 / (int)sizeof(T) : UNIT;
#endif
  static constexpr int GS = ((RAW + 4 * UNIT - 1) / (4 * UNIT)) * (4 * UNIT) + PAD;
  static constexpr int EVB = (((int)sizeof(GrpEvent<T, G::n>) + 127) / 128) * 128;
  static constexpr int SMEM = EVB + GPW * GS * (int)sizeof(T);
};

// Layout of the jamps in HBM between K1 and K2: X[event][listed combination][flow][8], the 8 = 2 (2 h_t + h_tbar) +
// re/im.  A warp of K2 reads 4 (fp64) or 2 x 4 (fp32) consecutive flows = 256 / 128 contiguous bytes per load.
template <class G> struct XGeom {
  static constexpr int NCOL = G::ncol, NT = NCOL / 8, NPAIR = NT * (NT + 1) / 2, GRP = NCOL * 8;
  static_assert(NCOL % 8 == 0, "tile geometry");
};

// Arguments of the three kernels of one chunk of events (pointers already offset to the chunk)
struct PipeArgs {
  LaunchArgs a;
  void* ev;                  // GrpEvent<T, N>[nevt]
  void* xt;                  // TC[nevt][ncombo][ncol][8] (+ one group of slack)
  const void* cfrag;         // 120 flows: C' in MMA fragment order (global memory), else unused
  int ncombo;                // gluon-helicity combinations with at least one good helicity row
  unsigned char combo[32];   // ... in increasing order
  unsigned char vmask[32];   // per listed combination: bit v = 2 h_t + h_tbar set iff that helicity row is good
};

// helicity row of gluon-helicity combination gg (bit N-1-i = gluon i) and variant v = 2 h_t + h_tbar
template <int N> __host__ __device__ __forceinline__ int grp_hel_of(int gg, int v) {
  constexpr int NPAR = N + 2;
  int h = 0;
#pragma unroll
  for (int i = 0; i < N; i++) {
    const int p = (i < 2) ? i : i + 2;
    h |= ((gg >> (N - 1 - i)) & 1) << (NPAR - 1 - p);
  }
  h |= (v >> 1) << (NPAR - 1 - 2);
  h |= (v & 1) << (NPAR - 1 - 3);
  return h;
}

// ------------------------------------------------------------------------------------------------------------------
// K0: per event, helicity-independent data.  Thread = (event, task); tasks: one per gluon subset, one per gluon
// (polarisation basis), six for the quark line (ubar(t), v(tbar), the four Q).  Every task reads the momenta it needs
// from global memory (incoming convention: +p for the initial, -p for the final state).
// ------------------------------------------------------------------------------------------------------------------
template <typename T, int N>
__global__ void __launch_bounds__(128) setup_kernel(const LaunchArgs a, GrpEvent<T, N>* __restrict__ evs) {
  constexpr int NPAR = N + 2, NSUB = 1 << N, NTASK = NSUB + N + 6, PT = (NTASK <= 32) ? 32 : 64;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long e = gid / PT;
  const int task = (int)(gid % PT);
  if (e >= a.nevt || task >= NTASK) return;
  GrpEvent<T, N>& ev = evs[e];
  const double* pm = a.mom + e * (NPAR * 4);
  auto kd = [&](int p, int c) { const double x = __ldg(pm + 4 * p + c); return (p < 2) ? x : -x; };
  const double mw = a.par.mt * a.par.wt;
  if (task < NSUB) {
    // gluon subset m: momentum sum, quark-line momentum after it, 1/K^2, quark-line denominator; invariants from
    // pairwise products 2 k_i.k_j in fp64 (never (sum k)^2, which cancels for collinear / soft gluons).
    // Branch-free: members are picked with 0/1 factors (exact)
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
    if (m == 0) ev.mt = T(a.par.mt);
  } else if (task < NSUB + N) {
    const int i = task - NSUB, p = (i < 2) ? i : i + 2;
    mom4<T> k;
    for (int c = 0; c < 4; c++) k.c[c] = T(kd(p, c));
    const polbasis<T> pb = make_polbasis<T>((p < 2) ? k : neg(k));
    for (int c = 0; c < 3; c++) { ev.pol[i][c] = pb.e1[c]; ev.pol[i][3 + c] = pb.e2[c]; }
  } else {
    // tasks 0,1: ubar(t), v(tbar) for both helicities; tasks 2..5: Q(h_t, h_tbar) = ubar gamma^mu v
    const int w = task - NSUB - N;
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

// ------------------------------------------------------------------------------------------------------------------
// K1 pieces
// ------------------------------------------------------------------------------------------------------------------
template <class G, typename T, typename TC> struct GrpWalkCtx;

// Colour-ordered gluon currents of one group, level by level (|seq| = 2 .. n).  One copy of the vertex code: the
// levels, the tasks of a level and the terms of a task are run-time loops over the generated tables (keeps the
// kernel small enough for the instruction cache; the loop bodies are ~100 FMA-pipe instructions each).
template <class G, typename T, typename TC, int LS>
__device__ __forceinline__ void grp_tree_level(const GrpEvent<T, G::n>& ev, T* slots, TC* X, int r, bool active, int Lrt) {
  // LS > 0: the level is a compile-time constant and the term loops are unrolled (straight-line task body: the
  // loads of later terms move above the arithmetic of earlier ones); LS == 0: run-time level Lrt, one copy of the code
  constexpr int LPG = GrpGeom<G, T>::LPG, UT = ME_UNROLL_T;
  const int L = LS ? LS : Lrt;
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
      TreeAcc<T> tacc;
      tacc.zero();
      T kt[4], kt2[4];   // momentum of the task's sequence and twice it
      {
        const T* q = ev.Ksub[(h0 >> 8) & 31u];
#pragma unroll
        for (int i = 0; i < 4; i++) { kt[i] = q[i]; kt2[i] = q[i] + q[i]; }
      }
      // Static levels: the three-gluon terms load every prefix seq[:m] (as A) and every suffix seq[m:] (as B) of the
      // sequence; the four-gluon term with split points (i, k) needs the prefix i, the suffix k and the middle block, so
      // it takes the first two from registers and loads only the middle one (9 instead of 15 operand loads per task
      // at the top level of n = 4: the tree is bound by shared-memory traffic). 
      constexpr bool CACHE = (LS > 2);
      constexpr bool SG = (G::signs != 0);   // operand words carry a sign (no twin slots): applied to A at every use
      constexpr int NC = (LS > 2) ? LS - 2 : 1;
      vec4<T> pre[NC], suf[NC];   // pre[m - 1] = Jord(seq[:m]), m = 1 .. L - 2;  suf[m - 2] = Jord(seq[m:]), m = 2 .. L - 1
      // run-time levels: the word of the next term is on its way while this term is evaluated (gg_ttggg fp64 +2.9 %,
      // mixed +2.7 %, fp32 +0.7 %, measured)
#ifdef ME_WORD_PREFETCH
      constexpr bool PREF = (LS == 0) && (ME_WORD_PREFETCH != 0);
#else
      constexpr bool PREF = (LS == 0);
#endif
      unsigned wq = PREF ? __ldg(tw + 2) : 0u;
      auto word = [&](int idx) {
        if constexpr (PREF) {
          const unsigned cur = wq;
          wq = __ldg(tw + 2 + min(idx + 1, W - 3));
          return cur;
        } else {
          return __ldg(tw + 2 + idx);
        }
      };
      auto term3 = [&](int j) {
        const unsigned w = word(j);
        ME_ASSERT((w & 255u) < (unsigned)G::nslot && ((w >> 8) & 255u) < (unsigned)G::nslot);
        const vec4<T> Ar = GrpSlot<T>::template ld<false>(slots, w & 255u, 0u);
        const vec4<T> B = GrpSlot<T>::ld(slots, (w >> 8) & 255u, 0u);
        if constexpr (CACHE) {
          const int m = j + 1;
          if (m <= LS - 2) pre[m - 1] = Ar;
          if (m >= 2) suf[m - 2] = B;
        }
        tacc.v3(SG ? vsgn(Ar, w >> 31) : Ar, B, ev.Ksub[(w >> 16) & 31u], kt, kt2);
      };
      auto term4 = [&](int j, int i, int k) {
        const unsigned w = word(NV3 + j);
        ME_ASSERT((w & 255u) < (unsigned)G::nslot && ((w >> 8) & 255u) < (unsigned)G::nslot && ((w >> 16) & 255u) < (unsigned)G::nslot);
        const vec4<T> B = GrpSlot<T>::ld(slots, (w >> 8) & 255u, 0u);
        if constexpr (CACHE) {
          tacc.v4(SG ? vsgn(pre[i - 1], w >> 31) : pre[i - 1], B, suf[k - 2]);
        } else {
          const vec4<T> A = GrpSlot<T>::template ld<(G::signs != 0)>(slots, w & 255u, w >> 31);
          const vec4<T> C = GrpSlot<T>::ld(slots, (w >> 16) & 255u, 0u);
          tacc.v4(A, B, C);
        }
      };
      if constexpr (LS > 0) {
        // term j of the three-gluon list splits the sequence after j + 1 gluons; the four-gluon list runs over the
        // split points (i, k), 1 <= i < k <= L - 1, in that order (emit_group.py level_table)
#pragma unroll
        for (int j = 0; j < LS - 1; j++) term3(j);
        int idx = 0;
#pragma unroll
        for (int i = 1; i < LS; i++)
#pragma unroll
          for (int k = i + 1; k < LS; k++) { term4(idx, i, k); idx++; }
      } else {
#pragma unroll(UT)
        for (int j = 0; j < NV3; j++) term3(j);
#pragma unroll(UT)
        for (int j = 0; j < NV4; j++) term4(j, 1, 2);
      }
      const vec4<T> acc = tacc.finish(ev.ik[(h0 >> 8) & 31u]);
      if (!TOP) {
        ME_ASSERT((h0 & 255u) < (unsigned)G::nslot && ((h0 >> 16) & 255u) < (unsigned)G::nslot);
        GrpSlot<T>::st(slots, h0 & 255u, acc);
        if (G::signs == 0 && ((h0 >> 16) & 255u)) {   // even length: the negated twin, for the reversed sequence
          vec4<T> nacc;
#pragma unroll
          for (int i = 0; i < 4; i++) nacc.c[i] = -acc.c[i];
          GrpSlot<T>::st(slots, (h0 >> 16) & 255u, nacc);
        }
      } else {
        // the full-length current is contracted at once with the four t-tbar currents: the j = 0 term of the
        // jamps of this sequence and of its reverse
        if constexpr (GrpInit<G>::GLOBAL) {
          // ... parked in the jamp buffer itself (rows of the two flows), where the leaves of the walk pick it
          // up: it stays in L2 until the leaf overwrites it with the finished jamp
          const unsigned h1 = __ldg(tw + 1);
          TC* ja = X + (h1 & 127u) * 8;
          TC* jb = X + ((h1 >> 8) & 127u) * 8;
          const T sb = (h1 >> 31) ? T(-1) : T(1);
#pragma unroll
          for (int v = 0; v < 4; v++) {
            const vec4<T> q = GrpVec<T>::ld(ev.Q[v], 0u);
            const cx<T> a = mdot(q, acc);
            GrpWalkCtx<G, T, TC>::st2(ja + 2 * v, TC(a.re), TC(a.im));
            GrpWalkCtx<G, T, TC>::st2(jb + 2 * v, TC(sb * a.re), TC(sb * a.im));
          }
        } else {
          // ... in "init" slot t of shared memory, read by the leaves of the walk
          // (stored like a current slot, chunk v = Q(v).J: same swizzle, same conflict pattern as the other slots)
          vec4<T> ini;
#pragma unroll
          for (int v = 0; v < 4; v++) ini.c[v] = mdot(GrpVec<T>::ld(ev.Q[v], 0u), acc);
          GrpSlot<T>::st(slots, G::nslot + t, ini);
        }
      }
    }
  }
  __syncwarp();
}

template <class G, typename T, typename TC, int LS>
__device__ __forceinline__ void grp_tree_static(const GrpEvent<T, G::n>& ev, T* slots, TC* X, int r, bool active) {
  grp_tree_level<G, T, TC, LS>(ev, slots, X, r, active, LS);
  if constexpr (LS < G::n) grp_tree_static<G, T, TC, LS + 1>(ev, slots, X, r, active);
}

template <class G, typename T, typename TC>
__device__ __forceinline__ void grp_tree(const GrpEvent<T, G::n>& ev, T* slots, TC* X, int r, bool active) {
  // one copy of the tree code per level with the term loops unrolled (n = 4: +2 % fp64, +5 % fp32, measured), or one
  // copy for all levels with run-time loops
  // (2: only the top level, which holds most of the tree's work, as a compile-time constant)
#ifdef ME_TREE_STATIC
  constexpr int STATIC = ME_TREE_STATIC;
#else
  // measured: n = 4 all levels static (+2 % fp64, +5 % fp32); n = 5 fp32 top level only (+4.8 %; all levels +2 %); n = 5
  // fp64 / mixed run-time levels (top level static -7 %, all static -28 %: 168 registers, 3200 instructions)
  constexpr int STATIC = (G::n <= 4) ? 1 : ((sizeof(T) == 4) ? 2 : 0);
#endif
  if constexpr (STATIC == 1) {
    grp_tree_static<G, T, TC, 2>(ev, slots, X, r, active);
  } else if constexpr (STATIC == 2) {
#pragma unroll 1
    for (int L = 2; L < G::n; L++) grp_tree_level<G, T, TC, 0>(ev, slots, X, r, active, L);
    grp_tree_level<G, T, TC, G::n>(ev, slots, X, r, active, G::n);
  } else {
#pragma unroll 1
    for (int L = 2; L <= G::n; L++) grp_tree_level<G, T, TC, 0>(ev, slots, X, r, active, L);
  }
}

// Quark-line walk of lane (s1[, h_t]): depth-first loop nest over the gluons that follow s1.  The words are read
// in execution order from the role's stream (emit_group.py role_stream); psi[j] = Psi(path[:j]) stays in registers.
template <class G, typename T, typename TC>
struct GrpWalkCtx {
  const GrpEvent<T, G::n>* ev;
  const T* slots;
  TC* X;  // jamps of this group in HBM: [ncol][8]
  const unsigned* stream;
  int ht;
  // one word of look-ahead in the role stream (padded by one word) for n = 5: +1 % fp32, +1.5 % mixed, measured
  static constexpr bool AHEAD = (G::n >= 5);
  unsigned ahead;
  __device__ __forceinline__ void start() { if constexpr (AHEAD) ahead = __ldg(stream++); }
  __device__ __forceinline__ unsigned next() {
    if constexpr (AHEAD) { const unsigned w = ahead; ahead = __ldg(stream++); return w; }
    else return __ldg(stream++);
  }
  __device__ __forceinline__ vec4<T> cur(unsigned w) const { ME_ASSERT((w & 255u) < (unsigned)G::nslot); return GrpSlot<T>::template ld<(G::signs != 0)>(slots, w & 255u, w >> 31); }
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
  // J_flow(h_t, b) = init + a  ->  X[flow][2 (2 h_t + b) + re/im]; stores bypass L1 (the table words live there)
  __device__ __forceinline__ static void st2(double* q, double x, double y) { __stcg(reinterpret_cast<double2*>(q), make_double2(x, y)); }
  __device__ __forceinline__ static void st2(float* q, float x, float y) { __stcg(reinterpret_cast<float2*>(q), make_float2(x, y)); }
  // finished jamps: read once by the colour kernel, so they leave L2 first (the per-event data of K0 and the parked
  // full-length currents stay)
  __device__ __forceinline__ static void stf(double* q, double x, double y) { __stcs(reinterpret_cast<double2*>(q), make_double2(x, y)); }
  __device__ __forceinline__ static void stf(float* q, float x, float y) { __stcs(reinterpret_cast<float2*>(q), make_float2(x, y)); }
  __device__ __forceinline__ static void ld2(const double* q, double& x, double& y) { const double2 t = __ldcg(reinterpret_cast<const double2*>(q)); x = t.x; y = t.y; }
  __device__ __forceinline__ static void ld2(const float* q, float& x, float& y) { const float2 t = __ldcg(reinterpret_cast<const float2*>(q)); x = t.x; y = t.y; }
  __device__ __forceinline__ void leaf(const spin4<PS> (&Xs)[WP::NCH], unsigned w) const {
    constexpr bool HTL = GrpGeom<G, T>::HTL;
    constexpr int NV = HTL ? 4 : 2;          // (h_t, b) values this lane completes: v = v0 + k
    const int f = (w >> 16) & 127;
    ME_ASSERT(f < G::ncol);
    const int v0 = HTL ? 0 : 2 * ht;
    TC* q = X + f * 8 + 2 * v0;
    T ini[NV][2];
    if constexpr (GrpInit<G>::GLOBAL) {
#pragma unroll
      for (int k = 0; k < NV; k++) { TC x, y; ld2(q + 2 * k, x, y); ini[k][0] = T(x); ini[k][1] = T(y); }
    } else {
      ME_ASSERT((w & 255u) >= (unsigned)G::nslot && (w & 255u) < (unsigned)(G::nslot + G::ninit));
      const T sg = (w >> 31) ? T(-1) : T(1);
      const vec4<T> iv = GrpSlot<T>::template ld<false>(slots, w & 255u, 0u);
#pragma unroll
      for (int k = 0; k < NV; k++) { ini[k][0] = sg * iv.c[v0 + k].re; ini[k][1] = sg * iv.c[v0 + k].im; }
    }
#pragma unroll
    for (int b = 0; b < 2; b++) {
      const spin4<T> vb = ld_spin<T>(ev->v[b]);
      spin4<PS> vw;
#pragma unroll
      for (int i = 0; i < 4; i++) vw.c[i] = mk<PS>(WP::widen(vb.c[i].re), WP::widen(vb.c[i].im));
#pragma unroll
      for (int c = 0; c < WP::NCH; c++) {
        const cx<PS> a = row_col(Xs[c], vw);
        fin(q, ini, HTL ? c : 0, b, a.re, a.im);
      }
    }
  }
  // finished jamp(s) of (chain c, b): packed pair = both h_t at once
  __device__ __forceinline__ static void fin(TC* q, const T (&ini)[GrpGeom<G, T>::HTL ? 4 : 2][2], int c, int b, f2 re, f2 im) {
    stf(q + 2 * b, TC(ini[b][0] + re.v.x), TC(ini[b][1] + im.v.x));                  // h_t = 0: v = b
    stf(q + 4 + 2 * b, TC(ini[2 + b][0] + re.v.y), TC(ini[2 + b][1] + im.v.y));      // h_t = 1: v = 2 + b
  }
  template <typename S>
  __device__ __forceinline__ static void fin(TC* q, const T (&ini)[GrpGeom<G, T>::HTL ? 4 : 2][2], int c, int b, S re, S im) {
    const int k = 2 * c + b;   // HTL: c = h_t; otherwise c = 0 and q already points at the lane's h_t
    stf(q + 2 * k, TC(ini[k][0] + re), TC(ini[k][1] + im));
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

// ------------------------------------------------------------------------------------------------------------------
// Quark-line walk of the fp32 build when a lane walks ONE t helicity (n = 5): every complex number is a packed
// (re, im) pair and a complex product c * z is accumulated as P += c.re * z, Q += c.im * z (sum = P + i Q): two FFMA2
// with a broadcast scalar and the pair as loaded, instead of four scalar FFMA.  That walk is bound by instruction
// issue (ncu: 66 % issue-active, FMA pipe 57 %), so halving its FP instructions is what helps.
// ------------------------------------------------------------------------------------------------------------------
struct sp2 { float2 c[4]; };              // spinor, components as (re, im)
struct spq { float2 P[4], Q[4]; };        // spinor being accumulated: component k = P[k] + i Q[k]
__device__ __forceinline__ float2 bc(float x) { return make_float2(x, x); }
__device__ __forceinline__ void c2_mul(float2& P, float2& Q, float2 r, float2 z) { P = __fmul2_rn(bc(r.x), z); Q = __fmul2_rn(bc(r.y), z); }
__device__ __forceinline__ void c2_mac(float2& P, float2& Q, float2 r, float2 z) { P = __ffma2_rn(bc(r.x), z, P); Q = __ffma2_rn(bc(r.y), z, Q); }
__device__ __forceinline__ void c2_msc(float2& P, float2& Q, float2 r, float2 z) { P = __ffma2_rn(bc(-r.x), z, P); Q = __ffma2_rn(bc(-r.y), z, Q); }
struct jcomb { float2 jp, jm, jt, jtb; };   // J0 + J3, J0 - J3, J1 + i J2, J1 - i J2
__device__ __forceinline__ jcomb c2_jcomb(const vec4<float>& J) {
  jcomb r;
  const float2 j0 = pk(J.c[0]), j1 = pk(J.c[1]), j3 = pk(J.c[3]);
  const float2 ij2 = make_float2(-J.c[2].im, J.c[2].re);
  r.jp = __fadd2_rn(j0, j3);
  r.jm = __fadd2_rn(j0, make_float2(-j3.x, -j3.y));
  r.jt = __fadd2_rn(j1, ij2);
  r.jtb = __fadd2_rn(j1, make_float2(-ij2.x, -ij2.y));
  return r;
}
// X = R Jslash  /  X += R Jslash   (me_ops.cuh row_slash / row_slash_add)
__device__ __forceinline__ void c2_slash(spq& X, const sp2& R, const jcomb& j) {
  c2_mul(X.P[0], X.Q[0], R.c[2], j.jp);  c2_mac(X.P[0], X.Q[0], R.c[3], j.jt);
  c2_mul(X.P[1], X.Q[1], R.c[2], j.jtb); c2_mac(X.P[1], X.Q[1], R.c[3], j.jm);
  c2_mul(X.P[2], X.Q[2], R.c[0], j.jm);  c2_msc(X.P[2], X.Q[2], R.c[1], j.jt);
  c2_mul(X.P[3], X.Q[3], R.c[1], j.jp);  c2_msc(X.P[3], X.Q[3], R.c[0], j.jtb);
}
__device__ __forceinline__ void c2_slash_add(spq& X, const sp2& R, const jcomb& j) {
  c2_mac(X.P[0], X.Q[0], R.c[2], j.jp);  c2_mac(X.P[0], X.Q[0], R.c[3], j.jt);
  c2_mac(X.P[1], X.Q[1], R.c[2], j.jtb); c2_mac(X.P[1], X.Q[1], R.c[3], j.jm);
  c2_mac(X.P[2], X.Q[2], R.c[0], j.jm);  c2_msc(X.P[2], X.Q[2], R.c[1], j.jt);
  c2_mac(X.P[3], X.Q[3], R.c[1], j.jp);  c2_msc(X.P[3], X.Q[3], R.c[0], j.jtb);
}
__device__ __forceinline__ sp2 c2_fold(const spq& X) {
  sp2 r;
#pragma unroll
  for (int k = 0; k < 4; k++) r.c[k] = fold_pq(X.P[k], X.Q[k]);
  return r;
}
// complex product r * z, folded
__device__ __forceinline__ float2 c2_prod(float2 r, float2 z) {
  float2 p, q;
  c2_mul(p, q, r, z);
  return fold_pq(p, q);
}
// X (qslash + m) gd   (me_ops.cuh row_prop): q real, gd complex
__device__ __forceinline__ sp2 c2_prop(const sp2& X, const float* q, float m, float2 gd) {
  const float qp = q[0] + q[3], qm = q[0] - q[3];
  const float2 qt = make_float2(q[1], q[2]), qtb = make_float2(q[1], -q[2]);
  float2 o[4];
  // o0 = m X0 + qp X2 + X3 qt;  o1 = m X1 + qm X3 + X2 qtb;  o2 = m X2 + qm X0 - X1 qt;  o3 = m X3 + qp X1 - X0 qtb
  o[0] = __fadd2_rn(__ffma2_rn(bc(qp), X.c[2], __fmul2_rn(bc(m), X.c[0])), c2_prod(X.c[3], qt));
  o[1] = __fadd2_rn(__ffma2_rn(bc(qm), X.c[3], __fmul2_rn(bc(m), X.c[1])), c2_prod(X.c[2], qtb));
  const float2 t2 = c2_prod(X.c[1], qt), t3 = c2_prod(X.c[0], qtb);
  o[2] = __fadd2_rn(__ffma2_rn(bc(qm), X.c[0], __fmul2_rn(bc(m), X.c[2])), make_float2(-t2.x, -t2.y));
  o[3] = __fadd2_rn(__ffma2_rn(bc(qp), X.c[1], __fmul2_rn(bc(m), X.c[3])), make_float2(-t3.x, -t3.y));
  sp2 r;
#pragma unroll
  for (int k = 0; k < 4; k++) r.c[k] = c2_prod(o[k], gd);
  return r;
}
__device__ __forceinline__ float2 c2_col(const sp2& X, const sp2& v) {
  float2 P, Q;
  c2_mul(P, Q, X.c[0], v.c[0]);
#pragma unroll
  for (int k = 1; k < 4; k++) c2_mac(P, Q, X.c[k], v.c[k]);
  return fold_pq(P, Q);
}
__device__ __forceinline__ sp2 c2_spin(const float* p) {
  const spin4<float> a = ld_spin<float>(p);
  sp2 r;
#pragma unroll
  for (int k = 0; k < 4; k++) r.c[k] = pk(a.c[k]);
  return r;
}

template <class G, typename TC, int D>
struct GrpWalkC2 {
  typedef GrpWalkCtx<G, float, TC> Ctx;
  __device__ __forceinline__ static void node(Ctx& c, sp2 (&psi)[G::n]) {
    const unsigned w0 = c.next();
    spq X;
    c2_slash(X, psi[0], c2_jcomb(c.cur(w0)));
#pragma unroll
    for (int j = 1; j < D; j++) c2_slash_add(X, psi[j], c2_jcomb(c.cur(c.next())));
    {
      const unsigned m = (w0 >> 8) & 31u;
      psi[D] = c2_prop(c2_fold(X), c.ev->qsub[m], c.ev->mt, make_float2(c.ev->gd[m][0], c.ev->gd[m][1]));
    }
#pragma unroll 1
    for (int child = 0; child < G::n - D; child++) GrpWalkC2<G, TC, D + 1>::node(c, psi);
  }
};
template <class G, typename TC>
struct GrpWalkC2<G, TC, G::n> {
  typedef GrpWalkCtx<G, float, TC> Ctx;
  __device__ __forceinline__ static void node(Ctx& c, sp2 (&psi)[G::n]) {
    spq X;
    c2_slash(X, psi[1], c2_jcomb(c.cur(c.next())));
#pragma unroll
    for (int j = 2; j < G::n; j++) c2_slash_add(X, psi[j], c2_jcomb(c.cur(c.next())));
    const unsigned w = c.next();
    // leaf: J_flow(h_t, b) = init + X . v(b), b = 0, 1
    const sp2 Xf = c2_fold(X);
    const int f = (w >> 16) & 127;
    ME_ASSERT(f < G::ncol);
    TC* q = c.X + f * 8 + 4 * c.ht;
    float ini[2][2];
    if constexpr (GrpInit<G>::GLOBAL) {
#pragma unroll
      for (int k = 0; k < 2; k++) { TC x, y; Ctx::ld2(q + 2 * k, x, y); ini[k][0] = float(x); ini[k][1] = float(y); }
    } else {
      const float sg = (w >> 31) ? -1.f : 1.f;
      const float* ji = c.slots + (w & 255u) * 8 + 4 * c.ht;
#pragma unroll
      for (int k = 0; k < 2; k++) { ini[k][0] = sg * ji[2 * k]; ini[k][1] = sg * ji[2 * k + 1]; }
    }
#pragma unroll
    for (int b = 0; b < 2; b++) {
      const float2 a = c2_col(Xf, c2_spin(c.ev->v[b]));
      Ctx::stf(q + 2 * b, TC(ini[b][0] + a.x), TC(ini[b][1] + a.y));
    }
  }
};

// ------------------------------------------------------------------------------------------------------------------
// K1: one warp per (event, unit); a unit is GPW listed gluon-helicity combinations, one per lane group.
// ------------------------------------------------------------------------------------------------------------------
template <class G, typename T, typename TC, int MINB>
__global__ void __launch_bounds__(32, MINB) amp_kernel(const PipeArgs p) {
  typedef GrpGeom<G, T> GE;
  constexpr int N = G::n, LPG = GE::LPG, GPW = GE::GPW;
  typedef GrpEvent<T, N> EV;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  EV& ev = *reinterpret_cast<EV*>(smem_raw);
  T* gbase = reinterpret_cast<T*>(smem_raw + GE::EVB);
  const int lane = threadIdx.x;
  const int gi = lane / LPG, r = lane - gi * LPG;
  const int nunit = (p.ncombo + GPW - 1) / GPW;
  T* slots = gbase + (size_t)((gi < GPW) ? gi : 0) * GE::GS;
#if defined(ME_CHECK) && ME_CHECK
  for (int i = lane; i < GPW * GE::GS; i += 32) gbase[i] = T(__longlong_as_double(0x7ff8000000000000ll));
  __syncwarp();
#endif
  // One warp per (event, unit).  (Persistent warps over a range of units measured 0-12 % slower: warps that start at
  // different times mix their tree and walk phases on the FP64 pipe, persistent ones run them in step.)
  {
    const long long e = blockIdx.x / nunit;
    const int unit = (int)(blockIdx.x - e * nunit);
    {
      // ---- a1: the event's helicity-independent data (K0), HBM -> shared memory past L1 (the table words live there)
      // (asynchronous 16-byte copies, all in flight at once: one round trip to L2 / HBM instead of one per loop pass)
      const char* src = reinterpret_cast<const char*>(reinterpret_cast<const EV*>(p.ev) + e);
      const unsigned dst = (unsigned)__cvta_generic_to_shared(&ev);
      static_assert(sizeof(EV) % 16 == 0, "GrpEvent is copied in 16-byte pieces");
#pragma unroll
      for (int i = lane; i < (int)(sizeof(EV) / 16); i += 32)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + 16u * (unsigned)i), "l"(src + 16 * i) : "memory");
      asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
    }
    __syncwarp();
    const int ci = unit * GPW + gi;                       // position in the list of combinations
    const bool active = (gi < GPW) && (ci < p.ncombo);
    const int grp = p.combo[active ? ci : 0];             // gluon-helicity combination
    // ---- a2: polarisation vectors of this group's gluon helicities
    if (active && r < N) {
      const int pp = (r < 2) ? r : r + 2;
      const int lam = ((grp >> (N - 1 - r)) & 1) ? 1 : -1;
      polbasis<T> pb;
      for (int c = 0; c < 3; c++) { pb.e1[c] = ev.pol[r][c]; pb.e2[c] = ev.pol[r][3 + c]; }
      GrpSlot<T>::st(slots, r, polvec(pb, lam, pp >= 2));
    }
    __syncwarp();
    // ---- a3: colour-ordered gluon currents, level by level; the full-length ones are contracted with Q
    grp_tree<G, T, TC>(ev, slots, reinterpret_cast<TC*>(p.xt) + ((size_t)e * p.ncombo + (active ? ci : 0)) * XGeom<G>::GRP, r, active);
    // ---- a3-a5: quark line; every leaf completes one jamp and stores it
    if (active) {
      typedef GrpWalkCtx<G, T, TC> Ctx;
      Ctx c;
      c.ev = &ev; c.slots = slots;
      c.X = reinterpret_cast<TC*>(p.xt) + ((size_t)e * p.ncombo + ci) * XGeom<G>::GRP;
      c.stream = G::role(GE::HTL ? r : (r >> 1));
      c.ht = GE::HTL ? 0 : (r & 1);
      c.start();
      // fp32 with one t helicity per lane (n = 5): the complex-packed walk (+2.4 %, measured)
#ifdef ME_WALK_C2
      constexpr bool C2 = (ME_WALK_C2 != 0) && sizeof(T) == 4 && !GE::HTL;
#else
      constexpr bool C2 = sizeof(T) == 4 && !GE::HTL;
#endif
      if constexpr (C2) {
        sp2 psi[G::n];
        psi[0] = c2_spin(ev.ub[c.ht]);
        GrpWalkC2<G, TC, 1>::node(c, psi);
      } else {
        spin4<typename Ctx::PS> psi[Ctx::WP::NCH][G::n];
#pragma unroll
        for (int h = 0; h < Ctx::WP::NCH; h++) psi[h][0] = c.psi0(h);
        GrpWalk<G, T, TC, 1>::node(c, psi);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
// K2 pieces
// ------------------------------------------------------------------------------------------------------------------
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

// D(8x8) += A(8x4) . B(4x8) in fp64 on the tensor cores (SASS: DMMA.8x8x4); thread t holds A[t/4][t%4], B[t%4][t/4],
// D[t/4][2 (t%4)], D[t/4][2 (t%4) + 1]
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
// D(16x8) += A(16x8) . B(8x8), TF32 inputs, fp32 accumulation (SASS: HMMA.1688.F32.TF32)
__device__ __forceinline__ void hmma1688(float (&d)[4], const unsigned (&a)[4], unsigned b0, unsigned b1) {
  asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ unsigned to_tf32(float x) {
  unsigned r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return r;
}


// ------------------------------------------------------------------------------------------------------------------
// K2: the colour contraction as tensor-core MMAs.  Per gluon-helicity combination, the 8 real vectors x_m (row m = 2
// (2 h_t + h_tbar) + re/im of X[flow][8]) give  q_m = sum_{I <= J} X_I C'_{IJ} . X_J  over the 8 x 8 tiles of C
// (C' = C with the diagonal tiles halved; the caller doubles the result: C is symmetric).
//   A fragment   thread (row = lane / 4, c = lane % 4) holds x_row at the flows 4 idx + c, idx < ncol / 4, loaded
//                straight from HBM (one 8- or 4-byte load per thread = 256 / 128 contiguous bytes per warp);
//   B fragment   C' from shared memory in fragment order; the columns of a tile are permuted, n -> flow
//                8 J + n / 2 + 4 (n % 2), so that the two D columns of a thread are flows 8 J + c and 8 J + c + 4:
//                flows whose x the thread already holds, and the row dot q_m += D . x needs no second load.
// ------------------------------------------------------------------------------------------------------------------
template <int NCOL, typename TC> struct ColFrag;

// C' entry: from shared memory, or (120 flows) from the fragment-ordered copy in global memory past L1 (the
// amplitude warps running beside the colour warps keep their table words there)
template <bool GLOBAL, typename V> __device__ __forceinline__ V cf_ld(const V* q) {
  if constexpr (GLOBAL) return __ldcg(q);
  else return *q;
}

// fp64: mma.sync m8n8k4 f64, one combination per tile; MMA row m = row of X[flow][8]
template <int NCOL> struct ColFrag<NCOL, double> {
  static constexpr int GPT = 1, NW = NCOL / 4, NT = NCOL / 8, JB = (NT < 5) ? NT : 5;
  static_assert(NT % JB == 0, "tile blocking");
  double a[NW];
  __device__ __forceinline__ void load(const double* X, int lane) {
    const double* p = X + (lane & 3) * 8 + (lane >> 2);
#pragma unroll
    for (int i = 0; i < NW; i++) a[i] = __ldcs(p + 32 * i);
  }
  // cf: [pair(I,J)][k-step s][lane]: B[k = lane % 4][n = lane / 4] = C'[8 I + 4 s + k][8 J + perm(n)]
  // returns the thread's part of q_m (m = lane / 4); the quad sum and the re + im sum are the caller's
  template <bool CFG> __device__ __forceinline__ double quad(const double* cf, int lane) const {
    double q = 0.0;
#pragma unroll
    for (int J0 = 0; J0 < NT; J0 += JB) {
      double d[JB][2];
#pragma unroll
      for (int j = 0; j < JB; j++) d[j][0] = d[j][1] = 0.0;
      // I outer, J inner: consecutive MMAs go to different accumulators
#pragma unroll
      for (int I = 0; I < J0 + JB; I++)
#pragma unroll
        for (int s = 0; s < 2; s++)
#pragma unroll
          for (int j = 0; j < JB; j++) {
            const int J = J0 + j;
            if (J >= I) dmma884(d[j][0], d[j][1], a[2 * I + s], cf_ld<CFG>(cf + ((J * (J + 1) / 2 + I) * 2 + s) * 32 + lane));
          }
#pragma unroll
      for (int j = 0; j < JB; j++) {
        q = ::fma(d[j][0], a[2 * (J0 + j)], q);
        q = ::fma(d[j][1], a[2 * (J0 + j) + 1], q);
      }
    }
    return q;
  }
  // w[idx] += |x|^2 of the flows 4 idx + c if the thread's row belongs to a good helicity (rows are added by the caller)
  __device__ __forceinline__ void weights(double (&w)[NW], bool keep) const {
#pragma unroll
    for (int i = 0; i < NW; i++) w[i] = keep ? ::fma(a[i], a[i], w[i]) : w[i];
  }
};

// fp32 / mixed: mma.sync m16n8k8 tf32, two combinations per tile.  Thread (g = lane / 4, c = lane % 4) owns the
// re and im rows of variant v = g % 4 of combination g / 4: MMA rows g and g + 8, one 8-byte load per flow.  X is
// split as hi + lo with hi = tf32(x), lo = tf32(x - hi): the integer colour numerators are exact in TF32, so every
// product carries fp32 accuracy and the sum accumulates in fp32
template <int NCOL> struct ColFrag<NCOL, float> {
  static constexpr int GPT = 2, NW = NCOL / 4, NT = NCOL / 8, JB = (NT < 5) ? NT : 5;
  static_assert(NT % JB == 0, "tile blocking");
  float x[NT][4];  // [k-block][a0: re row, flow 8 I + c; a1: im row, same flow; a2: re row, flow 8 I + c + 4; a3: im row]
  __device__ __forceinline__ void load(const float* X, int lane) {
    const int g = lane >> 2;
    const float* p = X + (g >> 2) * (NCOL * 8) + (lane & 3) * 8 + 2 * (g & 3);
#pragma unroll
    for (int I = 0; I < NT; I++) {
      const float2 u = __ldcs(reinterpret_cast<const float2*>(p + 64 * I));
      const float2 w = __ldcs(reinterpret_cast<const float2*>(p + 64 * I + 32));
      x[I][0] = u.x; x[I][1] = u.y; x[I][2] = w.x; x[I][3] = w.y;
    }
  }
  // cf: [pair(I,J)][lane][2]: b0 = C'[8 I + lane % 4][8 J + perm(lane / 4)], b1 = C'[8 I + lane % 4 + 4][...]
  // returns the thread's part of q_re + q_im of its variant
  template <bool CFG> __device__ __forceinline__ float quad(const float* cf, int lane) const {
    float q = 0.f;
#pragma unroll
    for (int J0 = 0; J0 < NT; J0 += JB) {
      float d[JB][4];
#pragma unroll
      for (int j = 0; j < JB; j++) d[j][0] = d[j][1] = d[j][2] = d[j][3] = 0.f;
#pragma unroll
      for (int I = 0; I < J0 + JB; I++) {
        unsigned ah[4], al[4];
#pragma unroll
        for (int i = 0; i < 4; i++) {
          ah[i] = to_tf32(x[I][i]);
          al[i] = to_tf32(x[I][i] - __uint_as_float(ah[i]));
        }
#pragma unroll
        for (int j = 0; j < JB; j++) {
          const int J = J0 + j;
          if (J >= I) {
            const float2 b = cf_ld<CFG>(reinterpret_cast<const float2*>(cf + ((J * (J + 1) / 2 + I) * 32 + lane) * 2));
            hmma1688(d[j], al, __float_as_uint(b.x), __float_as_uint(b.y));
            hmma1688(d[j], ah, __float_as_uint(b.x), __float_as_uint(b.y));
          }
        }
      }
#pragma unroll
      for (int j = 0; j < JB; j++) {
        q = fmaf(d[j][0], x[J0 + j][0], q); q = fmaf(d[j][1], x[J0 + j][2], q);
        q = fmaf(d[j][2], x[J0 + j][1], q); q = fmaf(d[j][3], x[J0 + j][3], q);
      }
    }
    return q;
  }
  __device__ __forceinline__ void weights(float (&w)[NW], bool keep) const {
#pragma unroll
    for (int I = 0; I < NT; I++) {
      w[2 * I] = keep ? fmaf(x[I][1], x[I][1], fmaf(x[I][0], x[I][0], w[2 * I])) : w[2 * I];
      w[2 * I + 1] = keep ? fmaf(x[I][3], x[I][3], fmaf(x[I][2], x[I][2], w[2 * I + 1])) : w[2 * I + 1];
    }
  }
};

template <class G, typename TC> struct ColGeom {
  // 24 flows: C' is 1.5-3 KB, so a block is ONE warp with a few KB of shared memory and < 3 K registers: such blocks
  // become resident beside the amplitude warps of the following chunk and run under them (high-priority stream).
  // 120 flows: C' is 30-61 KB in shared memory, shared by the 8 warps of a block.  (A copy in global memory read by
  // one-warp blocks was measured: 4.6 TB/s of L2 traffic in fp32, the amplitude kernel beside it 20 % slower.)
#ifndef ME_K2_WARPS
#define ME_K2_WARPS 8   // warps per block for 120 flows.  Round 3, gg_ttggg 262144 events, (warps per block, colour warps per
#endif                  // SM) = (8, 8) / (4, 4) / (4, 8) / (16, 16): fp64 242.2 / 243.2 / 241.7 / 246.4 ms, fp32 113.4 / 113.4 /
#ifndef ME_K2_WPS       // 112.4 / 123.3 ms: within 1 % except the last, (8, 8) kept
#define ME_K2_WPS 8
#endif
  static constexpr int WARPS = (G::ncol <= 24) ? 1 : ME_K2_WARPS;
  static constexpr bool CF_GLOBAL = false;
  static constexpr int WPS = (G::ncol <= 24) ? 32 : ME_K2_WPS;   // colour warps per SM (grid sizing; 4, 8, 16, 32 measured)
  static constexpr int GPT = ColFrag<G::ncol, TC>::GPT, NCOL = G::ncol;
  static constexpr int CF = XGeom<G>::NPAIR * 64;                        // TC elements of C' in fragment order
  static constexpr int PERW = (int)sizeof(double) * ((1 << (G::n + 2)) + NCOL);   // per warp: |M_h|^2, colour weights
  static constexpr int SMEM = (CF_GLOBAL ? 0 : CF * (int)sizeof(TC)) + WARPS * PERW;
};

// C' (diagonal tiles halved, tile columns permuted) in MMA fragment order; CM::at16(i): entry i of the row-major
// integer colour numerators (global memory)
template <class G, typename TC, class CM>
__device__ __forceinline__ TC cfrag_entry(int i) {
  constexpr int GPT = ColFrag<G::ncol, TC>::GPT, NCOL = G::ncol;
  const int pair = i >> 6;
  int ca, n;
  if (GPT == 1) { const int l = i & 31, s = (i >> 5) & 1; ca = 4 * s + (l & 3); n = l >> 2; }
  else { const int l = (i >> 1) & 31; ca = (l & 3) + 4 * (i & 1); n = l >> 2; }
  int J = 0;
  while ((J + 1) * (J + 2) / 2 <= pair) J++;
  const int I = pair - J * (J + 1) / 2;
  const int cb = (n >> 1) + 4 * (n & 1);
  const TC cv = TC(CM::at16((8 * I + ca) * NCOL + 8 * J + cb));
  return (I == J) ? TC(0.5) * cv : cv;
}
template <class G, typename TC, class CM>
__global__ void cfrag_kernel(TC* out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < ColGeom<G, TC>::CF) out[i] = cfrag_entry<G, TC, CM>(i);
}

// K2: one warp per event (the warps stride over the events of the chunk).
template <class G, typename TC, class CM, int MODE>
__global__ void __launch_bounds__(ColGeom<G, TC>::WARPS * 32) colour_kernel(const PipeArgs p) {
  typedef ColGeom<G, TC> CG;
  typedef ColFrag<G::ncol, TC> Frag;
  constexpr int N = G::n, NPAR = N + 2, NCOMB = 1 << NPAR, NCOL = G::ncol, GPT = CG::GPT, NW = Frag::NW;
  constexpr bool CFG = CG::CF_GLOBAL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr size_t CFB = CFG ? 0 : CG::CF * sizeof(TC);
  double* mh = reinterpret_cast<double*>(smem_raw + CFB + (size_t)warp * CG::PERW);  // [NCOMB]
  double* wcs = mh + NCOMB;                                                          // [NCOL]
  const LaunchArgs& a = p.a;
  const TC* cf;
  if constexpr (CFG) {
    cf = reinterpret_cast<const TC*>(p.cfrag);
  } else {
    TC* cfs = reinterpret_cast<TC*>(smem_raw);
    for (int i = tid; i < CG::CF; i += CG::WARPS * 32) cfs[i] = cfrag_entry<G, TC, CM>(i);
    __syncthreads();
    cf = cfs;
  }
  const long long wstride = (long long)gridDim.x * CG::WARPS;
  const long long w0 = (long long)blockIdx.x * CG::WARPS + warp;
  const int ntile = (p.ncombo + GPT - 1) / GPT;
  const TC* xbase = reinterpret_cast<const TC*>(p.xt);
  auto tile_ptr = [&](long long e, int ti) { return xbase + ((size_t)e * p.ncombo + (size_t)ti * GPT) * XGeom<G>::GRP; };
  auto is_good = [&](int h) { return MODE == MODE_FILTER || ((a.good.mask[h >> 6] >> (h & 63)) & 1ull) != 0ull; };
  Frag cur, nxt;
  if (w0 < a.nevt) cur.load(tile_ptr(w0, 0), lane);
  for (long long e = w0; e < a.nevt; e += wstride) {
    for (int h = lane; h < NCOMB; h += 32) mh[h] = 0.0;
    TC wacc[NW];
#pragma unroll
    for (int i = 0; i < NW; i++) wacc[i] = TC(0);
    __syncwarp();
#pragma unroll 1
    for (int ti = 0; ti < ntile; ti++) {
      // the next tile (of this event or of the warp's next event) is on its way while this one is contracted
      const bool more_here = ti + 1 < ntile;
      const long long en = more_here ? e : e + wstride;
      if (en < a.nevt) nxt.load(tile_ptr(en, more_here ? ti + 1 : 0), lane);
      // ---- a6 on the tensor cores
      TC q = cur.template quad<CFG>(cf, lane);
      q += __shfl_xor_sync(0xffffffffu, q, 1);
      q += __shfl_xor_sync(0xffffffffu, q, 2);   // MMA row(s) of the quad complete
      int ci, v;                                  // listed combination and variant of this thread's row(s)
      if constexpr (GPT == 1) {
        q += __shfl_xor_sync(0xffffffffu, q, 4);  // re + im rows of variant v = lane / 8
        ci = ti; v = lane >> 3;
        if ((lane & 7) == 0) mh[grp_hel_of<N>(p.combo[ci], v)] = 2.0 * q;
      } else {
        ci = 2 * ti + (lane >> 4); v = (lane >> 2) & 3;   // the thread's rows are re and im of one variant
        if ((lane & 3) == 0 && ci < p.ncombo) mh[grp_hel_of<N>(p.combo[ci], v)] = (double)(2.f * q);
      }
      if (MODE == MODE_SELECT && a.selcol) {
        // a8 colour weights: |J_c|^2 of the good (h_t, h_tbar) rows, per thread for its row(s); rows are added below
        cur.weights(wacc, ci < p.ncombo && ((p.vmask[ci < p.ncombo ? ci : 0] >> v) & 1));
      }
      cur = nxt;
    }
    __syncwarp();
    // ---- a7-a9 for this event
    if (MODE == MODE_FILTER) {
      double total = 0.0;
      for (int h = 0; h < NCOMB; h++) total += mh[h];
      for (int h = lane; h < NCOMB; h += 32) {
        const double f = (total > 0.0) ? mh[h] / total : 0.0;
        atomicMax(a.fracmax + h, (unsigned long long)__double_as_longlong(f));
      }
    } else {
      {
        // helicity sum in table order (a7), ME (a9) and helicity selection (a8): in-order scan
        constexpr int PER = NCOMB / 32;
        double val[PER];
        bool ok[PER];
#pragma unroll
        for (int i = 0; i < PER; i++) {
          const int h = lane * PER + i;
          ok[i] = is_good(h);
          val[i] = ok[i] ? mh[h] : 0.0;
        }
        double total;
        int sel;
        grp_warp_select<PER>(val, ok, (MODE == MODE_SELECT && a.selhel) ? a.rndhel[e] : 0.0, lane, total, sel);
        if (lane == 0) {
          const double g = a.gs[e];
          a.me[e] = total * ipow<2 * N>(g) * (1.0 / (double(G::denom) * double(G::cden)));
          if (MODE == MODE_SELECT && a.selhel) a.selhel[e] = sel;
        }
      }
      if (MODE == MODE_SELECT && a.selcol) {
        // rows 0..7 of the warp hold partial weights of the same flows: add them, lanes 0..3 publish flow 4 idx + c
#pragma unroll
        for (int i = 0; i < NW; i++) {
          TC w = wacc[i];
          w += __shfl_xor_sync(0xffffffffu, w, 4);
          w += __shfl_xor_sync(0xffffffffu, w, 8);
          w += __shfl_xor_sync(0xffffffffu, w, 16);
          if (lane < 4) wcs[4 * i + lane] = (double)w;
        }
        __syncwarp();
        // multichannel (reading R17): flows the event's channel does not contribute to are not selectable
        const unsigned* cfl = a.channel ? a.chanflows + 4 * min(max(a.channel[e], 0), a.nchan - 1) : nullptr;
        constexpr int PER = (NCOL + 31) / 32;
        double val[PER];
        bool ok[PER];
#pragma unroll
        for (int i = 0; i < PER; i++) {
          const int c = lane * PER + i;
          ok[i] = c < NCOL && (!cfl || ((cfl[c >> 5] >> (c & 31)) & 1u));
          val[i] = ok[i] ? wcs[c] : 0.0;
        }
        double total;
        int sel;
        grp_warp_select<PER>(val, ok, a.rndcol[e], lane, total, sel);
        if (lane == 0) a.selcol[e] = sel;
      }
    }
    __syncwarp();
  }
}

}  // namespace me
