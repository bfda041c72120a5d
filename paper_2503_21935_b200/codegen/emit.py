"""CUDA source emitter: turns a diagrams.Structure into csrc/gen/proc_<name>.cuh.

The emitted struct has (all force-inlined, templated on the arithmetic type T):
  Event<T>           per-event, helicity-independent data (momenta, polarisation / spinor bases,
                     propagator denominators formed in fp64 from the fp64 inputs)
  setup(p, par, ev)  fills Event from momenta[npar][4]
  jamps(ev, h, J)    colour-flow amplitudes J[ncol] of helicity row h, coupling stripped (g = 1)
and the constant tables (colour-matrix numerators, denominator, counts).
Layout "B0": one event per thread, one helicity per loop trip, straight-line code.
"""
from __future__ import annotations

import itertools

from . import diagrams


def _nm(prefix, legs):
    return prefix + "_" + "_".join(str(x) for x in legs)


class Emitter:
    def __init__(self, name: str, st: diagrams.Structure):
        self.name, self.st = name, st
        self.lines = []
        self.ind = 0

    def w(self, s=""):
        self.lines.append("  " * self.ind + s if s else "")

    # ------------------------------------------------------------------ event-level data
    def gluon_subsets(self):
        g = self.st.gluons
        return [s for r in range(2, len(g) + 1) for s in itertools.combinations(g, r)]

    def prefix_subsets(self):
        g = self.st.gluons
        return [s for r in range(1, len(g)) for s in itertools.combinations(g, r)]

    def emit_event_struct(self):
        st = self.st
        self.w("template <typename T> struct Event {")
        self.ind += 1
        self.w(f"me::mom4<T> k[{st.npar}];  // incoming-convention momenta: +p (initial), -p (final)")
        self.w(f"me::polbasis<T> pol[{st.npar}];  // gluon legs only")
        self.w("me::spin4<T> ub[2], v[2];  // ubar(t), v(tbar) for helicity -1 / +1")
        for s in self.gluon_subsets():
            self.w(f"T {_nm('ik', s)};  // 1 / K_S^2")
        for s in self.prefix_subsets():
            self.w(f"me::cx<T> {_nm('gd', s)};  // 1 / (q^2 - m^2 + i m Gamma), q = p_t - K_S")
        self.w("T mt;")
        self.ind -= 1
        self.w("};")

    def emit_setup(self):
        st = self.st
        self.w("// p: momenta[npar][4] of one event (fp64, E px py pz); invariants are formed in fp64 from")
        self.w("// pairwise products 2 k_i.k_j so that collinear/soft denominators do not cancel (DESIGN.md).")
        self.w("template <typename T, typename LOAD> ME_HD static void setup(LOAD p, const me::DevParams& par, Event<T>& ev) {")
        self.w("const double mt = par.mt, wt = par.wt;")
        self.ind += 1
        self.w(f"double kd[{st.npar}][4];")
        self.w(f"for (int i = 0; i < {st.npar}; i++)")
        self.w("  for (int m = 0; m < 4; m++) { double x = p(i, m); kd[i][m] = (i < 2) ? x : -x; ev.k[i].c[m] = T(kd[i][m]); }")
        self.w(f"double d2[{st.npar}][{st.npar}];  // 2 k_i . k_j")
        self.w(f"for (int i = 0; i < {st.npar}; i++)")
        self.w(f"  for (int j = i + 1; j < {st.npar}; j++)")
        self.w("    d2[i][j] = 2.0 * (kd[i][0] * kd[j][0] - kd[i][1] * kd[j][1] - kd[i][2] * kd[j][2] - kd[i][3] * kd[j][3]);")
        for g in st.gluons:
            sign = "" if g < 2 else "me::neg"
            self.w(f"ev.pol[{g}] = me::make_polbasis<T>({sign}(ev.k[{g}]));")
        self.w("{")
        self.w("  me::spinbasis<T> sb = me::make_spinbasis<T>(me::neg(ev.k[2]), T(mt));")
        self.w("  ev.ub[0] = me::bar(me::spinor_u(sb, -1)); ev.ub[1] = me::bar(me::spinor_u(sb, +1));")
        self.w("  sb = me::make_spinbasis<T>(me::neg(ev.k[3]), T(mt));")
        self.w("  ev.v[0] = me::spinor_v(sb, -1); ev.v[1] = me::spinor_v(sb, +1);")
        self.w("}")
        for s in self.gluon_subsets():
            terms = " + ".join(f"d2[{a}][{b}]" for a, b in itertools.combinations(s, 2))
            self.w(f"ev.{_nm('ik', s)} = T(1.0 / ({terms}));")
        self.w("const double mw = mt * wt;")
        for s in self.prefix_subsets():
            # (k_t + K_S)^2 - m^2 = 2 k_t.K_S + K_S^2
            terms = [f"d2[{min(2, a)}][{max(2, a)}]" for a in s]
            terms += [f"d2[{a}][{b}]" for a, b in itertools.combinations(s, 2)]
            self.w("{ const double den = " + " + ".join(terms) + "; const double n = 1.0 / (den * den + mw * mw);")
            self.w(f"  ev.{_nm('gd', s)} = me::mk<T>(T(den * n), T(-mw * n)); }}")
        self.w("ev.mt = T(mt);")
        self.ind -= 1
        self.w("}")

    # ------------------------------------------------------------------ per-helicity amplitudes
    def ksum(self, legs):
        """Expression for K_S (mom4<T>) as a local variable name; emitted on first use."""
        legs = tuple(legs)
        if len(legs) == 1:
            return f"ev.k[{legs[0]}]"
        name = _nm("K", legs)
        if name not in self.kdone:
            self.kdone.add(name)
            sub = self.ksum(legs[:-1])
            self.w(f"const me::mom4<T> {name} = {sub} + ev.k[{legs[-1]}];")
        return name

    def emit_jamps(self):
        st = self.st
        self.kdone = set()
        self.w("// colour-flow amplitudes of helicity row h (particle 0 = most significant bit), g = 1")
        self.w("template <typename T> ME_HD static void jamps(const Event<T>& ev, int h, me::cx<T>* J) {")
        self.ind += 1
        for g in st.gluons:
            out = "false" if g < 2 else "true"
            self.w(f"const me::vec4<T> t{st.trees_on[(g,)][0]} = me::polvec(ev.pol[{g}], "
                   f"((h >> {st.npar - 1 - g}) & 1) ? 1 : -1, {out});")
        self.w(f"const me::spin4<T> psi0 = me::select(((h >> {st.npar - 1 - 2}) & 1) != 0, ev.ub[1], ev.ub[0]);")
        self.w(f"const me::spin4<T> vv = me::select(((h >> {st.npar - 1 - 3}) & 1) != 0, ev.v[1], ev.v[0]);")
        # gluon trees
        done_groups = set()
        for t in st.trees:
            if t.kind == "leaf":
                continue
            ik = "ev." + _nm("ik", t.legs)
            if t.kind == "v3":
                a, b = t.children
                ka, kb = self.ksum(st.trees[a].legs), self.ksum(st.trees[b].legs)
                self.w(f"const me::vec4<T> t{t.tid} = me::vvv_current(t{a}, t{b}, {ka}, {kb}, {ik});")
            elif t.group not in done_groups:
                done_groups.add(t.group)
                a, b, c = t.children
                self.w(f"me::vec4<T> t{t.tid}, t{t.tid + 1}, t{t.tid + 2};")
                self.w(f"me::vvvv_currents(t{a}, t{b}, t{c}, {ik}, t{t.tid}, t{t.tid + 1}, t{t.tid + 2});")
        # ordered currents
        for seq, terms in st.ordered.items():
            expr = ""
            for c, tid in terms:
                expr += (" + " if c > 0 else " - ") + f"t{tid}"
            expr = expr[3:] if expr.startswith(" + ") else "me::zero_vec4<T>()" + expr
            self.w(f"const me::vec4<T> {_nm('o', seq)} = {expr};")
        # quark line, depth first over ordered prefixes
        self.dfs((), ["psi0"])
        self.ind -= 1
        self.w("}")

    def ordered_ref(self, seq):
        if len(seq) == 1:
            return f"t{self.st.trees_on[(seq[0],)][0]}", 1
        can, sgn = diagrams.canonical(seq)
        return _nm("o", can), sgn

    def dfs(self, prefix, stack):
        """stack[j] = name of Psi(prefix[:j]) for j = 0..len(prefix)."""
        st = self.st
        for g in st.gluons:
            if g in prefix:
                continue
            seq = prefix + (g,)
            self.w("{")
            self.ind += 1
            # X = sum_j Psi(seq[:j]) . Jord-slash(seq[j:])
            for j in range(len(seq)):
                cur, sgn = self.ordered_ref(seq[j:])
                if j == 0:
                    self.w(f"me::spin4<T> X = me::row_slash{'' if sgn > 0 else '_neg'}({stack[0]}, {cur});")
                else:
                    self.w(f"me::row_slash_{'add' if sgn > 0 else 'sub'}(X, {stack[j]}, {cur});")
            if len(seq) == st.ngl:
                self.w(f"J[{st.flows.index(seq)}] = me::row_col(X, vv);")
            else:
                name = _nm("psi", seq)
                legs = tuple(sorted(seq))
                # q = p_t - K_S = -(k_t + K_S)
                ks = self.ksum_q(legs)
                self.w(f"const me::spin4<T> {name} = me::row_prop(X, {ks}, ev.mt, ev.{_nm('gd', legs)});")
                self.dfs(seq, stack + [name])
            self.ind -= 1
            self.w("}")

    def ksum_q(self, legs):
        name = _nm("q", legs)
        if name not in self.kdone:
            # emitted inline at first use inside a scope: recompute each time (cheap, keeps scopes simple)
            pass
        expr = "me::neg(ev.k[2]" + "".join(f" + ev.k[{a}]" for a in legs) + ")"
        return expr

    # ------------------------------------------------------------------ whole file
    def emit(self):
        st = self.st
        self.w(f"// GENERATED by paper_2503_21935_b200/codegen (emit.py) -- do not edit.  Process {self.name}:")
        self.w(f"// g g -> t tbar + {st.ngl - 2} g, {st.ndiag} Feynman diagrams, {len(st.flows)} colour flows.")
        self.w("#pragma once")
        self.w('#include "../me_ops.cuh"')
        self.w('#include "../me_params.cuh"')
        self.w(f"struct Proc_{self.name} {{")
        self.ind += 1
        self.w(f"static constexpr int npar = {st.npar}, ncomb = {1 << st.npar}, ncol = {len(st.flows)}, "
               f"ngl = {st.ngl}, ndiag = {st.ndiag}, denom = {st.denom}, cden = {st.cmat_den};")
        self.emit_event_struct()
        self.emit_setup()
        self.emit_jamps()
        self.ind -= 1
        self.w("};")
        return "\n".join(self.lines) + "\n"


def tables(st: diagrams.Structure):
    """Constant tables as C initialisers: colour matrix numerators (int), flows."""
    n = len(st.flows)
    cm = ", ".join(str(st.cmat_num[i][j]) for i in range(n) for j in range(n))
    fl = ", ".join(str(x) for f in st.flows for x in f)
    return cm, fl


class EmitterDY(Emitter):
    """g ubar -> tau+ tau- + (n-1) g + ubar (diagrams.build_dy): the same one-event-per-thread layout.

    The quark line runs from the outgoing ubar (column spinor v, last particle) to the incoming ubar (row spinor vbar,
    particle 1), massless; besides the gluon blocks it carries ONE electroweak insertion, the photon / Z with its tau
    pair.  In the phase-stripped rules the insertion is a colourless leaf whose "polarisation" depends on the chirality
    X of the quark line:  W_X = sum_Y A_XY J_Y,  J_Y = ubar(tau-) gamma^mu P_Y v(tau+),
    A_XY = e^2 Qu Qtau / s + g_X^u g_Y^tau / (s - MZ^2 + i MZ GZ), applied as R -> R Wslash_L P_L + R Wslash_R P_R
    (me::row_slash_chiral).  With Psi0 / Psi1 the line prefixes without / with the insertion,
        Psi0(seq) = [ sum_j Psi0(seq[:j]) Jord-slash(seq[j:]) ] prop(q0),
        Psi1(seq) = [ sum_j Psi1(seq[:j]) Jord-slash(seq[j:]) + Psi0(seq) Wslash ] prop(q1),   Psi1() = vbar Wslash prop,
        J_sigma   = [ sum_j Psi1(sigma[:j]) Jord-slash(sigma[j:]) + Psi0(sigma) Wslash ] . v
    which reproduces every Feynman diagram of the CPU checker's enumeration (boson at every place of the line) once.
    """
    ROW, LEPP, LEPM = 1, 2, 3   # incoming ubar, tau+, tau-

    def col_leg(self):
        return self.st.npar - 1

    def all_subsets(self, lo):
        g = self.st.gluons
        return [s for r in range(lo, len(g) + 1) for s in itertools.combinations(g, r)]

    def emit_event_struct(self):
        st = self.st
        self.w("template <typename T> struct Event {")
        self.ind += 1
        self.w(f"me::mom4<T> k[{st.npar}];  // incoming-convention momenta: +p (initial), -p (final)")
        self.w(f"me::polbasis<T> pol[{st.npar}];  // gluon legs only")
        self.w("me::spin4<T> ub[2], v[2];    // vbar(ubar in), v(ubar out) for helicity -1 / +1")
        self.w("me::spin4<T> lub[2], lv[2];  // ubar(tau-), v(tau+)")
        self.w("me::cx<T> aLL, aLR, aRL, aRR;  // A_XY: X = chirality of the quark line, Y = of the lepton line")
        for s in self.all_subsets(2):
            self.w(f"T {_nm('ik', s)};  // 1 / K_S^2")
        for s in self.all_subsets(1):
            self.w(f"T {_nm('gd0', s)};  // 1 / q^2, q = -(k_ubar + K_S)")
        for s in self.all_subsets(0)[:-1]:
            self.w(f"T {_nm('gd1', s) if s else 'gd1_none'};  // 1 / q^2, q = -(k_ubar + K_S + k_tau+ + k_tau-)")
        self.ind -= 1
        self.w("};")

    def emit_setup(self):
        st = self.st
        R, LP, LM, C = self.ROW, self.LEPP, self.LEPM, self.col_leg()
        self.w("// p: momenta[npar][4] of one event (fp64, E px py pz); every invariant is formed in fp64 from the pairwise")
        self.w("// products 2 k_i.k_j (all particles are massless here).")
        self.w("template <typename T, typename LOAD> ME_HD static void setup(LOAD p, const me::DevParams& par, Event<T>& ev) {")
        self.ind += 1
        self.w(f"double kd[{st.npar}][4];")
        self.w(f"for (int i = 0; i < {st.npar}; i++)")
        self.w("  for (int m = 0; m < 4; m++) { double x = p(i, m); kd[i][m] = (i < 2) ? x : -x; ev.k[i].c[m] = T(kd[i][m]); }")
        self.w(f"double d2[{st.npar}][{st.npar}];  // 2 k_i . k_j")
        self.w(f"for (int i = 0; i < {st.npar}; i++)")
        self.w(f"  for (int j = i + 1; j < {st.npar}; j++)")
        self.w("    d2[i][j] = 2.0 * (kd[i][0] * kd[j][0] - kd[i][1] * kd[j][1] - kd[i][2] * kd[j][2] - kd[i][3] * kd[j][3]);")
        for g in st.gluons:
            sign = "" if g < 2 else "me::neg"
            self.w(f"ev.pol[{g}] = me::make_polbasis<T>({sign}(ev.k[{g}]));")
        self.w("{")
        self.w(f"  me::spinbasis<T> sb = me::make_spinbasis<T>(ev.k[{R}], T(0));")
        self.w("  ev.ub[0] = me::bar(me::spinor_v(sb, -1)); ev.ub[1] = me::bar(me::spinor_v(sb, +1));")
        self.w(f"  sb = me::make_spinbasis<T>(me::neg(ev.k[{C}]), T(0));")
        self.w("  ev.v[0] = me::spinor_v(sb, -1); ev.v[1] = me::spinor_v(sb, +1);")
        self.w(f"  sb = me::make_spinbasis<T>(me::neg(ev.k[{LM}]), T(0));")
        self.w("  ev.lub[0] = me::bar(me::spinor_u(sb, -1)); ev.lub[1] = me::bar(me::spinor_u(sb, +1));")
        self.w(f"  sb = me::make_spinbasis<T>(me::neg(ev.k[{LP}]), T(0));")
        self.w("  ev.lv[0] = me::spinor_v(sb, -1); ev.lv[1] = me::spinor_v(sb, +1);")
        self.w("}")
        self.w("{")
        self.w(f"  const double s = d2[{LP}][{LM}], dr = s - par.mz * par.mz, di = par.mz * par.wz, n = 1.0 / (dr * dr + di * di);")
        self.w("  const double zr = dr * n, zi = -di * n, ph = -(2.0 / 3.0) * par.ee2 / s;   // Qu Qtau = -2/3")
        self.w("  ev.aLL = me::mk<T>(T(ph + par.glu * par.gl * zr), T(par.glu * par.gl * zi));")
        self.w("  ev.aLR = me::mk<T>(T(ph + par.glu * par.gr * zr), T(par.glu * par.gr * zi));")
        self.w("  ev.aRL = me::mk<T>(T(ph + par.gru * par.gl * zr), T(par.gru * par.gl * zi));")
        self.w("  ev.aRR = me::mk<T>(T(ph + par.gru * par.gr * zr), T(par.gru * par.gr * zi));")
        self.w("}")

        def pairs(legs):
            return " + ".join(f"d2[{min(a, b)}][{max(a, b)}]" for a, b in itertools.combinations(legs, 2))
        for s in self.all_subsets(2):
            self.w(f"ev.{_nm('ik', s)} = T(1.0 / ({pairs(s)}));")
        for s in self.all_subsets(1):
            self.w(f"ev.{_nm('gd0', s)} = T(1.0 / ({pairs((R,) + s)}));")
        for s in self.all_subsets(0)[:-1]:
            self.w(f"ev.{_nm('gd1', s) if s else 'gd1_none'} = T(1.0 / ({pairs((R, LP, LM) + s)}));")
        self.ind -= 1
        self.w("}")

    def emit_jamps(self):
        st = self.st
        self.kdone = set()
        hb = lambda k: f"((h >> {st.npar - 1 - k}) & 1)"
        self.w("// colour-flow amplitudes of helicity row h (particle 0 = most significant bit), g_s = 1, for a quark line of")
        self.w("// chirality CH (two-component form, me::wsp): CH = 0 the row spinor lives in components (2,3), CH = 1 in (0,1)")
        self.w("template <int CH, typename T> ME_HD static void jamps_ch(const Event<T>& ev, int h, me::cx<T>* J) {")
        self.ind += 1
        for g in st.gluons:
            out = "false" if g < 2 else "true"
            self.w(f"const me::vec4<T> t{st.trees_on[(g,)][0]} = me::polvec(ev.pol[{g}], {hb(g)} ? 1 : -1, {out});")
        self.w(f"const me::wsp<T> psi0 = me::w_half<CH>(me::select({hb(self.ROW)} != 0, ev.ub[1], ev.ub[0]));")
        self.w(f"const me::spin4<T> vv = me::select({hb(self.col_leg())} != 0, ev.v[1], ev.v[0]);")
        self.w("me::vec4<T> W;  // the electroweak insertion seen by this chirality of the quark line")
        self.w("{")
        self.w("  me::vec4<T> lR, lL;")
        self.w(f"  me::chiral_currents(me::select({hb(self.LEPM)} != 0, ev.lub[1], ev.lub[0]), "
               f"me::select({hb(self.LEPP)} != 0, ev.lv[1], ev.lv[0]), lR, lL);")
        self.w("  const me::cx<T> aR = CH ? ev.aRR : ev.aLR, aL = CH ? ev.aRL : ev.aLL;")
        self.w("  for (int i = 0; i < 4; i++) W.c[i] = me::fma(aR, lR.c[i], aL * lL.c[i]);")
        self.w("}")
        done_groups = set()
        for t in st.trees:
            if t.kind == "leaf":
                continue
            ik = "ev." + _nm("ik", t.legs)
            if t.kind == "v3":
                a, b = t.children
                ka, kb = self.ksum(st.trees[a].legs), self.ksum(st.trees[b].legs)
                self.w(f"const me::vec4<T> t{t.tid} = me::vvv_current(t{a}, t{b}, {ka}, {kb}, {ik});")
            elif t.group not in done_groups:
                done_groups.add(t.group)
                a, b, c = t.children
                self.w(f"me::vec4<T> t{t.tid}, t{t.tid + 1}, t{t.tid + 2};")
                self.w(f"me::vvvv_currents(t{a}, t{b}, t{c}, {ik}, t{t.tid}, t{t.tid + 1}, t{t.tid + 2});")
        for seq, terms in st.ordered.items():
            expr = ""
            for c, tid in terms:
                expr += (" + " if c > 0 else " - ") + f"t{tid}"
            expr = expr[3:] if expr.startswith(" + ") else "me::zero_vec4<T>()" + expr
            self.w(f"const me::vec4<T> {_nm('o', seq)} = {expr};")
        self.w(f"const me::wsp<T> psi1 = me::w_prop<CH>(me::w_slash<CH>(psi0, W), {self.qexpr((), True)}, ev.gd1_none);")
        self.dfs_dy((), ["psi0"], ["psi1"])
        self.ind -= 1
        self.w("}")
        self.w("// an incoming antiquark of helicity +1 is carried by the components (2,3) of its row spinor vbar")
        self.w("template <typename T> ME_HD static void jamps(const Event<T>& ev, int h, me::cx<T>* J) {")
        self.w(f"  if ({hb(self.ROW)}) jamps_ch<0, T>(ev, h, J);")
        self.w("  else jamps_ch<1, T>(ev, h, J);")
        self.w("}")

    def qexpr(self, legs, with_boson):
        extra = f" + ev.k[{self.LEPP}] + ev.k[{self.LEPM}]" if with_boson else ""
        return f"me::neg(ev.k[{self.ROW}]" + "".join(f" + ev.k[{a}]" for a in legs) + extra + ")"

    def dfs_dy(self, prefix, s0, s1):
        """s0[j] / s1[j] = names of Psi0(prefix[:j]) / Psi1(prefix[:j])."""
        st = self.st
        for g in st.gluons:
            if g in prefix:
                continue
            seq = prefix + (g,)
            legs = tuple(sorted(seq))
            self.w("{")
            self.ind += 1
            for which, stack in (("X0", s0), ("X1", s1)):
                for j in range(len(seq)):
                    cur, sgn = self.ordered_ref(seq[j:])
                    if j == 0:
                        self.w(f"me::wsp<T> {which} = me::w_slash{'' if sgn > 0 else '_neg'}<CH>({stack[0]}, {cur});")
                    else:
                        self.w(f"me::w_slash_{'add' if sgn > 0 else 'sub'}<CH>({which}, {stack[j]}, {cur});")
            n0 = _nm("psi0", seq)
            self.w(f"const me::wsp<T> {n0} = me::w_prop<CH>(X0, {self.qexpr(legs, False)}, ev.{_nm('gd0', legs)});")
            self.w(f"X1 = X1 + me::w_slash<CH>({n0}, W);")
            if len(seq) == st.ngl:
                self.w(f"J[{st.flows.index(seq)}] = me::w_col<CH>(X1, vv);")
            else:
                n1 = _nm("psi1", seq)
                self.w(f"const me::wsp<T> {n1} = me::w_prop<CH>(X1, {self.qexpr(legs, True)}, ev.{_nm('gd1', legs)});")
                self.dfs_dy(seq, s0 + [n0], s1 + [n1])
            self.ind -= 1
            self.w("}")

    def emit(self):
        st = self.st
        self.w(f"// GENERATED by paper_2503_21935_b200/codegen (emit.py, EmitterDY) -- do not edit.  Process {self.name}:")
        self.w(f"// g ubar -> tau+ tau- + {st.ngl - 1} g + ubar (photon + Z), {st.ndiag} Feynman diagrams, {len(st.flows)} colour flows.")
        self.w("#pragma once")
        self.w('#include "../me_ops.cuh"')
        self.w('#include "../me_params.cuh"')
        self.w(f"struct Proc_{self.name} {{")
        self.ind += 1
        self.w(f"static constexpr int npar = {st.npar}, ncomb = {1 << st.npar}, ncol = {len(st.flows)}, "
               f"ngl = {st.ngl}, ndiag = {st.ndiag}, denom = {st.denom}, cden = {st.cmat_den};")
        self.emit_event_struct()
        self.emit_setup()
        self.emit_jamps()
        self.ind -= 1
        self.w("};")
        return "\n".join(self.lines) + "\n"
