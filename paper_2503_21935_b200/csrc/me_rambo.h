// me_rambo.h -- arguments of the device-side input generator (me_rambo.cu), called from me_api.cu.
#pragma once
namespace me {
struct RamboArgs {
  double* mom;      // [nevt][npar][4]
  double* gs;       // [nevt] or null
  double* rndhel;   // [nevt] or null
  double* rndcol;   // [nevt] or null
  double* weight;   // [nevt] phase-space weight or null
  long long nevt, start;
  double sqrts, alphas;  // alphas > 0: fixed; <= 0: alpha_s ~ U[0.10, 0.13] per event
  double mass[5];
  double wt0;
  int massive;
  unsigned long long key[4];
};
// returns a cudaError_t value
int launch_rambo(RamboArgs a, int nfin, unsigned long long seed, void* stream);
}  // namespace me
