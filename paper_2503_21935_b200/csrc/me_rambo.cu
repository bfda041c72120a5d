// me_rambo.cu -- device-side seeded inputs (the role of the paper's standalone
// application, "random numbers are drawn ... converted into particle momenta using a phase space sampling
// algorithm"): counter-based uniforms -> RAMBO flat phase space -> momenta[nevt][npar][4], plus the
// per-event g_s and the two selection randoms, written straight into HBM so that a batch never touches the host.
// Checked against the numpy oracle oracle/rambo.py, which implements the same counter-based generator and the same
// RAMBO steps on its own (tests/test_gpu_rambo.py: uniforms bit-exact, momenta and weights to rounding); no code is
// shared.  One event per thread.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "../../include/me_b200.h"
#include "me_rambo.h"

namespace {

__host__ __device__ inline unsigned long long splitmix64(unsigned long long x) {
  unsigned long long z = x + 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
// uniform in (0,1): a pure function of (key(seed, stream), index)
__device__ inline double uniform(unsigned long long key, unsigned long long idx) {
  unsigned long long x = splitmix64(idx ^ key);
  x = splitmix64(x + key);
  return ((double)(x >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

template <int NFIN>
__global__ void __launch_bounds__(128) rambo_kernel(me::RamboArgs a) {
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= a.nevt) return;
  const unsigned long long ge = (unsigned long long)(a.start + e);
  const double w = a.sqrts, pi = 3.14159265358979323846;
  // massless generation
  double q[NFIN][4], qs[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
  for (int i = 0; i < NFIN; i++) {
    const unsigned long long base = ge * (NFIN * 4) + 4 * i;
    const double r0 = uniform(a.key[0], base), r1 = uniform(a.key[0], base + 1), r2 = uniform(a.key[0], base + 2),
                 r3 = uniform(a.key[0], base + 3);
    const double c = 2.0 * r0 - 1.0, s = sqrt(1.0 - c * c), phi = 2.0 * pi * r1, f = -log(r2 * r3);
    q[i][0] = f; q[i][1] = f * s * cos(phi); q[i][2] = f * s * sin(phi); q[i][3] = f * c;
#pragma unroll
    for (int m = 0; m < 4; m++) qs[m] += q[i][m];
  }
  // conformal boost to the centre-of-mass frame
  const double mq = sqrt(qs[0] * qs[0] - qs[1] * qs[1] - qs[2] * qs[2] - qs[3] * qs[3]);
  const double b[3] = {-qs[1] / mq, -qs[2] / mq, -qs[3] / mq};
  const double x = w / mq, g = qs[0] / mq, aa = 1.0 / (1.0 + g);
  double p[NFIN][4];
#pragma unroll
  for (int i = 0; i < NFIN; i++) {
    const double bq = b[0] * q[i][1] + b[1] * q[i][2] + b[2] * q[i][3];
    p[i][0] = x * (g * q[i][0] + bq);
#pragma unroll
    for (int m = 0; m < 3; m++) p[i][1 + m] = x * (q[i][1 + m] + b[m] * q[i][0] + (aa * bq) * b[m]);
  }
  double wt = a.wt0;
  if (a.massive) {
    // xi-rescaling: sum_i sqrt(m_i^2 + xi^2 E_i^2) = w by Newton iteration
    double msum = 0.0;
#pragma unroll
    for (int i = 0; i < NFIN; i++) msum += a.mass[i];
    double xi = sqrt(1.0 - (msum / w) * (msum / w));
    for (int it = 0; it < 50; it++) {
      double f0 = -w, g0 = 0.0;
#pragma unroll
      for (int i = 0; i < NFIN; i++) {
        const double en = sqrt(a.mass[i] * a.mass[i] + xi * xi * p[i][0] * p[i][0]);
        f0 += en;
        g0 += xi * p[i][0] * p[i][0] / en;
      }
      const double dxi = f0 / g0;
      xi -= dxi;
      if (fabs(dxi) < 1e-15) break;
    }
    double ksum = 0.0, kprod = 1.0, k2e = 0.0;
#pragma unroll
    for (int i = 0; i < NFIN; i++) {
      const double k = xi * p[i][0], en = sqrt(a.mass[i] * a.mass[i] + k * k);
      ksum += k; kprod *= k / en; k2e += k * k / en;
      p[i][0] = en;
#pragma unroll
      for (int m = 1; m < 4; m++) p[i][m] *= xi;
    }
    double pw = 1.0;
    for (int i = 0; i < 2 * NFIN - 3; i++) pw *= ksum / w;
    wt = wt * pw * kprod * w / k2e;
  }
  double* o = a.mom + e * ((NFIN + 2) * 4);
  const double eb = 0.5 * w;
  o[0] = eb; o[1] = 0.0; o[2] = 0.0; o[3] = eb;
  o[4] = eb; o[5] = 0.0; o[6] = 0.0; o[7] = -eb;
#pragma unroll
  for (int i = 0; i < NFIN; i++)
#pragma unroll
    for (int m = 0; m < 4; m++) o[8 + 4 * i + m] = p[i][m];
  if (a.weight) a.weight[e] = wt;
  if (a.gs) a.gs[e] = (a.alphas > 0.0) ? sqrt(4.0 * pi * a.alphas) : sqrt(4.0 * pi * (0.10 + 0.03 * uniform(a.key[1], ge)));
  if (a.rndhel) a.rndhel[e] = uniform(a.key[2], ge);
  if (a.rndcol) a.rndcol[e] = uniform(a.key[3], ge);
}

}  // namespace

namespace me {

int launch_rambo(RamboArgs a, int nfin, unsigned long long seed, void* stream) {
  for (int s = 0; s < 4; s++) a.key[s] = splitmix64(seed * 0xD1342543DE82EF95ull + (unsigned long long)(s + 1));
  const double pi = 3.14159265358979323846;
  double fact1 = 1.0, fact2 = 1.0;
  for (int k = 2; k <= nfin - 1; k++) fact1 *= k;
  for (int k = 2; k <= nfin - 2; k++) fact2 *= k;
  a.wt0 = pow(pi / 2.0, nfin - 1) * pow(a.sqrts, 2 * nfin - 4) / (fact1 * fact2) * pow(2.0 * pi, 4 - 3 * nfin);
  a.massive = 0;
  for (int i = 0; i < nfin; i++) a.massive |= (a.mass[i] != 0.0);
  if (a.nevt == 0) return 0;
  const unsigned blocks = (unsigned)((a.nevt + 127) / 128);
  cudaStream_t st = (cudaStream_t)stream;
  switch (nfin) {
    case 2: rambo_kernel<2><<<blocks, 128, 0, st>>>(a); break;
    case 3: rambo_kernel<3><<<blocks, 128, 0, st>>>(a); break;
    case 4: rambo_kernel<4><<<blocks, 128, 0, st>>>(a); break;
    case 5: rambo_kernel<5><<<blocks, 128, 0, st>>>(a); break;
    default: return (int)cudaErrorInvalidValue;
  }
  return (int)cudaGetLastError();
}

}  // namespace me
