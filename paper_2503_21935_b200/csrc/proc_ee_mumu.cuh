// proc_ee_mumu.cuh -- e+ e- -> mu+ mu- through an s-channel photon and Z (2 diagrams, 1 colour,
// 16 helicities; BASELINE.json configs[0]).  Hand-written (the generator covers the gg processes).
//
//   M = sum_{X,Y in {L,R}} A_XY  [vbar(e+) g^mu P_X u(e-)] [ubar(mu-) g_mu P_Y v(mu+)],
//   A_XY = e^2/s + g_X g_Y / (s - MZ^2 + i MZ GZ)          (massless leptons)
// In the chiral representation P_L / P_R pick the upper / lower two spinor components, so the four
// chirality amplitudes are products of two-component currents (me::chiral_currents).
// Particles: 0 = e+ (in), 1 = e- (in), 2 = mu+ (out), 3 = mu- (out).
#pragma once
#include "me_ops.cuh"
#include "me_params.cuh"

struct Proc_ee_mumu {
  static constexpr int npar = 4, ncomb = 16, ncol = 1, ngl = 0, ndiag = 2, denom = 4, cden = 1;
  template <typename T> struct Event {
    me::spin4<T> vb[2], u[2], v[2], ub[2];  // vbar(e+), u(e-), v(mu+), ubar(mu-) for helicity -1 / +1
    me::cx<T> aRR, aRL, aLR, aLL;           // A_XY, X = electron line, Y = muon line
  };
  template <typename T, typename LOAD> ME_HD static void setup(LOAD p, const me::DevParams& par, Event<T>& ev) {
    me::mom4<T> k[4];
    double q[4];
    for (int m = 0; m < 4; m++) {
      q[m] = p(0, m) + p(1, m);
      for (int i = 0; i < 4; i++) k[i].c[m] = T(p(i, m));
    }
    const double s = q[0] * q[0] - q[1] * q[1] - q[2] * q[2] - q[3] * q[3];
    me::spinbasis<T> sb = me::make_spinbasis<T>(k[0], T(0));
    ev.vb[0] = me::bar(me::spinor_v(sb, -1)); ev.vb[1] = me::bar(me::spinor_v(sb, +1));
    sb = me::make_spinbasis<T>(k[1], T(0));
    ev.u[0] = me::spinor_u(sb, -1); ev.u[1] = me::spinor_u(sb, +1);
    sb = me::make_spinbasis<T>(k[2], T(0));
    ev.v[0] = me::spinor_v(sb, -1); ev.v[1] = me::spinor_v(sb, +1);
    sb = me::make_spinbasis<T>(k[3], T(0));
    ev.ub[0] = me::bar(me::spinor_u(sb, -1)); ev.ub[1] = me::bar(me::spinor_u(sb, +1));
    // Z propagator 1/(s - MZ^2 + i MZ GZ) and photon e^2/s, in fp64
    const double dr = s - par.mz * par.mz, di = par.mz * par.wz;
    const double n = 1.0 / (dr * dr + di * di);
    const double zr = dr * n, zi = -di * n;
    const double ph = par.ee2 / s;
    ev.aRR = me::mk<T>(T(ph + par.gr * par.gr * zr), T(par.gr * par.gr * zi));
    ev.aLL = me::mk<T>(T(ph + par.gl * par.gl * zr), T(par.gl * par.gl * zi));
    ev.aRL = me::mk<T>(T(ph + par.gr * par.gl * zr), T(par.gr * par.gl * zi));
    ev.aLR = ev.aRL;
  }
  template <typename T> ME_HD static void jamps(const Event<T>& ev, int h, me::cx<T>* J) {
    me::vec4<T> eR, eL, mR, mL;
    me::chiral_currents(me::select((h & 8) != 0, ev.vb[1], ev.vb[0]), me::select((h & 4) != 0, ev.u[1], ev.u[0]), eR, eL);
    me::chiral_currents(me::select((h & 1) != 0, ev.ub[1], ev.ub[0]), me::select((h & 2) != 0, ev.v[1], ev.v[0]), mR, mL);
    me::cx<T> a = ev.aRR * me::mdot(eR, mR);
    a = me::fma(ev.aLL, me::mdot(eL, mL), a);
    a = me::fma(ev.aRL, me::mdot(eR, mL), a);
    a = me::fma(ev.aLR, me::mdot(eL, mR), a);
    J[0] = a;
  }
};
#define ME_CMAT_EE_MUMU {1}
#define ME_FLOWS_EE_MUMU {0}
