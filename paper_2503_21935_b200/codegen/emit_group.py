"""Emitter for the "lane-group" kernel layout (csrc/me_group.cuh): csrc/gen/grp_<name>.cuh.

Layout: one CUDA block per event; a *group* of 2n lanes of one warp owns one
combination of the n gluon helicities; the helicities of t and tbar are handled inside the group, so
the gluon currents are computed once per gluon-helicity combination and shared by the four
(h_t, h_tbar) combinations.  Within a group

  * the colour-ordered gluon currents Jord(seq) are built level by level
    (length 2, 3, ...), one canonical sequence per lane, from a table of (slot, slot, momentum,
    sign) words: Jord(seq) = 1/K^2 [ sum_j V3(Jord(seq[:j]), Jord(seq[j:])) + sum_{i<j} V4(...)];
  * lane (s1, h_t) walks the quark line (steps a3-a5) for the flows that start with gluon s1: the walk
    is the same straight-line code for every s1 up to a relabelling of the gluons, so it is emitted
    once in *relative* labels (0 = s1, 1.. = the other gluons in increasing order) and each lane
    translates relative sequence ids to shared-memory slots through its role's table.

Everything here is index bookkeeping; the arithmetic lives in csrc/me_ops.cuh / me_group.cuh.
"""
from __future__ import annotations

import itertools


def canonical(seq):
    """(representative of {seq, reversed seq}, sign): Jord(rev) = (-1)^(len+1) Jord(seq)."""
    seq = tuple(seq)
    if len(seq) == 1 or seq[0] < seq[-1]:
        return seq, 1
    return tuple(reversed(seq)), (-1) ** (len(seq) + 1)


def mask_of(seq):
    m = 0
    for i in seq:
        m |= 1 << i
    return m


class Group:
    def __init__(self, name: str, n: int, twins=None):
        self.name, self.n = name, n
        # twins: every stored current of even length (the only ones whose reversed sequence carries a minus sign) is
        # stored twice, as +J and -J, and the tables point at the copy with the right sign: no sign handling at the
        # loads (8 integer instructions per loaded current).  Worth its shared memory for n = 4 (6 extra slots of 22);
        # for n = 5 (70 extra slots of 105) shared memory is what bounds the resident warps, so the sign bit stays.
        self.twins = (n <= 4) if twins is None else twins
        idx = tuple(range(n))
        self.flows = list(itertools.permutations(idx))
        self.flow_index = {f: i for i, f in enumerate(self.flows)}
        # slots: canonical sequences of length 1 .. n-1 (the full-length currents are contracted at once)
        self.slot = {}
        self.level_seqs = {}
        for L in range(1, n + 1):
            seqs = [s for c in itertools.combinations(idx, L) for s in itertools.permutations(c)
                    if canonical(s)[0] == s]
            self.level_seqs[L] = seqs
            if L < n:
                for s in seqs:
                    self.slot[s] = len(self.slot)
        self.twin = {}
        if self.twins:
            for s, i in list(self.slot.items()):
                if len(s) % 2 == 0:
                    self.twin[s] = len(self.slot) + len(self.twin)
        self.nslot = len(self.slot) + len(self.twin)
        assert self.nslot < 255 and len(self.flows) <= 128

    def ref(self, seq):
        can, sgn = canonical(seq)
        if sgn < 0 and can in self.twin:
            return self.twin[can], 1
        return self.slot[can], sgn

    # ------------------------------------------------------------------ gluon-current task tables
    def level_table(self, L):
        """Words per task: [header0, header1, v3 terms (L-1), v4 terms ((L-1)(L-2)/2)]."""
        words = []
        for seq in self.level_seqs[L]:
            top = L == self.n
            h0 = (255 if top else self.slot[seq]) | (mask_of(seq) << 8) | (self.twin.get(seq, 0) << 16)
            h1 = 0
            if top:
                rev = tuple(reversed(seq))
                rs = (-1) ** (L + 1)
                h1 = self.flow_index[seq] | (self.flow_index[rev] << 8) | ((1 << 31) if rs < 0 else 0)
            words += [h0, h1]
            for j in range(1, L):
                a, b = seq[:j], seq[j:]
                (sa, ga), (sb, gb) = self.ref(a), self.ref(b)
                words.append(sa | (sb << 8) | (mask_of(a) << 16) | (mask_of(b) << 21) | ((1 << 31) if ga * gb < 0 else 0))
            for i in range(1, L):
                for j in range(i + 1, L):
                    a, b, c = seq[:i], seq[i:j], seq[j:]
                    (sa, ga), (sb, gb), (sc, gc) = self.ref(a), self.ref(b), self.ref(c)
                    words.append(sa | (sb << 8) | (sc << 16) | ((1 << 31) if ga * gb * gc < 0 else 0))
        return words

    # ------------------------------------------------------------------ quark-line walk, relative labels
    def role_stream(self, s1):
        """Words consumed, in execution order, by the lanes whose first gluon is s1 (me_group.cuh GrpWalk).

        The walk is a depth-first loop nest over the gluons that follow s1 (relative labels 1.. = the other
        gluons in increasing order); a node with path (s1, p1..pk) consumes
          inner node: [path word: slot+sign of Jord(path), subset mask], then Jord(path[j:]) for j = 1..k
          leaf      : Jord(path[j:]) for j = 1..n-1 (the j = 0 block was contracted in the tree phase),
                      then [flow word: flow index << 16 | slot of the contracted full-length current (nslot + its
                      task index in the top level) | sign of Jord(path) relative to the canonical sequence]
        word bits: 0-7 slot, 8-12 subset mask, 16-22 flow, 31 sign."""
        n = self.n
        others = [i for i in range(n) if i != s1]
        out = []

        def cur_word(seq):
            slot, sgn = self.ref(seq)
            return slot | (mask_of(seq) << 8) | ((1 << 31) if sgn < 0 else 0)

        def node(path):
            if len(path) == n:
                for j in range(1, n):
                    out.append(cur_word(path[j:]))
                can, sgn = canonical(path)
                init = self.nslot + self.level_seqs[n].index(can)
                assert init < 256
                out.append((self.flow_index[path] << 16) | (mask_of(path) << 8) | init | ((1 << 31) if sgn < 0 else 0))
                return
            out.append(cur_word(path))
            for j in range(1, len(path)):
                out.append(cur_word(path[j:]))
            for g in others:
                if g not in path:
                    node(path + (g,))

        node((s1,))
        return out

    # ------------------------------------------------------------------ whole file
    def emit(self, cmat_num, cmat_den, ndiag, denom):
        n = self.n
        out = []
        o = out.append
        o(f"// GENERATED by paper_2503_21935_b200/codegen (emit_group.py) -- do not edit.  Process {self.name}:")
        o(f"// g g -> t tbar + {n - 2} g in the lane-group layout; {self.nslot} current slots, {len(self.flows)} flows.")
        o("#pragma once")
        o('#include "../me_ops.cuh"')
        for L in range(2, n + 1):
            tab = self.level_table(L)
            o(f"__device__ const unsigned int kGrpLevel{L}_{self.name}[] = {{{', '.join(str(x) for x in tab)}}};")
        roles = []
        for s1 in range(n):
            st = self.role_stream(s1)
            nstream = len(st)
            roles += st
        roles.append(0)   # one word of padding: the walk may read one word ahead of the last role's stream
        o(f"__device__ const unsigned int kGrpRole_{self.name}[] = {{{', '.join(str(x) for x in roles)}}};")
        o(f"struct Grp_{self.name} {{")
        o(f"  static constexpr int n = {n}, npar = {n + 2}, ncomb = {1 << (n + 2)}, ncol = {len(self.flows)}, "
          f"ndiag = {ndiag}, denom = {denom}, cden = {cmat_den}, nslot = {self.nslot}, ninit = {len(self.level_seqs[n])}, "
          f"signs = {0 if self.twins else 1}, "
          f"nstream = {nstream};")
        o("  __device__ __forceinline__ static const unsigned int* level(int L) {")
        o("    switch (L) {")
        for L in range(2, n + 1):
            o(f"      case {L}: return kGrpLevel{L}_{self.name};")
        o("    }")
        o("    return nullptr;")
        o("  }")
        o("  __device__ __forceinline__ static int ntask(int L) {")
        o("    switch (L) {")
        for L in range(2, n + 1):
            o(f"      case {L}: return {len(self.level_seqs[L])};")
        o("    }")
        o("    return 0;")
        o("  }")
        o(f"  __device__ __forceinline__ static const unsigned int* role(int s1) {{ return kGrpRole_{self.name} + s1 * {nstream}; }}")
        o("};")
        return "\n".join(out) + "\n"

    # ------------------------------------------------------------------ FLOP accounting (FMA = 2)
    def flops(self):
        """Algorithmic FLOPs of this layout per gluon-helicity combination (4 helicities) and per event."""
        n = self.n
        # per-op counts derived line by line from me_group.cuh (v3_acc, v4_acc) and me_ops.cuh (row_slash, row_slash_add,
        # row_prop, row_col, mdot): complex multiply 6, complex fma 8, real*complex fma 4
        # (V3: 30 + 8 + 8 for the three Minkowski products, 16 for the momentum combinations from kA and the task's
        # total momentum, 4 x 24 for the update; + 4 per task for twice the total momentum)
        V3, V4, SL, SLA, PROP, COL, DOT = 158, 188, 64, 72, 82, 30, 30
        tree = 0
        for L in range(2, n + 1):
            nt = len(self.level_seqs[L])
            tree += nt * ((L - 1) * V3 + (L - 1) * (L - 2) // 2 * V4 + 8 + 4)
        tree += len(self.level_seqs[n]) * (4 * DOT + 8)
        walk = 0
        rest = n - 1
        for k in range(1, n + 1):
            nodes = 1
            for i in range(k - 1):
                nodes *= rest - i
            terms = k - 1 if k == n else k
            per = SL + (terms - 1) * SLA + (2 * COL + 4 if k == n else PROP)
            walk += nodes * per
        walk *= 2 * n  # lanes (s1, h_t)
        ncol = len(self.flows)
        colour = 4 * (2 * ncol * (ncol + 1) + 2)
        return {"per_gluon_combination": tree + walk + colour, "tree": tree, "walk": walk, "colour": colour,
                "combinations": 1 << n, "per_event": 8 * (n + 2) * (n + 1) // 2 + 40 * (n + 2) + 30 * (1 << n) + 4 * 60}
