// me_params.cuh -- physics parameters as the kernels see them (filled by me_create from me_params).
#pragma once
namespace me {
struct DevParams {
  double mt, wt, mz, wz;
  double ee2, gl, gr;  // e^2 and the Z couplings g_L, g_R of the charged leptons (ee_mumu only)
};
}  // namespace me
