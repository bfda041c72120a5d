// me_params.cuh -- physics parameters as the kernels see them (filled by me_create from me_params).
#pragma once
namespace me {
struct DevParams {
  double mt, wt, mz, wz;
  double ee2, gl, gr;  // e^2 and the Z couplings g_L, g_R of the charged leptons
  double glu, gru;     // Z couplings of the up quark (Q = 2/3, T3 = 1/2)
};
}  // namespace me
