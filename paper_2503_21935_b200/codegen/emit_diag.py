"""Emitter for the diagram-by-diagram kernel (csrc/me_diag.cuh): csrc/gen/diag_<name>.cuh.

Multichannel support: the single-diagram-enhancement weight of channel d is
|A_d|^2 / sum_d' |A_d'|^2 with A_d the value of ONE Feynman diagram.  The matrix-element kernels never form single
diagrams (they work with colour-ordered currents), so this weight has its own, table-driven kernel; this module
enumerates the diagrams of g g -> t tbar + (n-2) g from diagrams.Structure and writes the tables:

  tree tasks    every gluon tree that is not a leaf (three-gluon vertex of two sub-trees, or one colour-structure term
                of a four-gluon vertex of three), level = number of legs: each tree current is computed once per
                helicity and shared by all the diagrams that contain it;
  chain tasks   quark-line prefixes (ordered lists of attached trees) with their trailing propagator, level = number of
                attached trees: shared by all the diagrams that start with the prefix;
  closures      (prefix, last tree) = one (term of a) diagram, with its channel.

Channel numbering (reading R17): the structural key of a diagram is the "|"-joined keys of the trees on
the quark line from t to tbar; a leaf's key is its particle index, a three-gluon vertex "(A,B)" with the lowest leg in
A, a four-gluon vertex "[A,B,C]" with the lowest leg in A and the lowest of the rest in B.  Channels are the distinct
keys in increasing byte order; the three terms of a four-gluon vertex share a key, hence a channel.  The CPU checker
builds the same numbering on its own from the same written rule; tests compare the two key lists.
"""
from __future__ import annotations

import itertools

from . import colour, diagrams


class Diagrams:
    def __init__(self, name: str, st: diagrams.Structure):
        self.name, self.st = name, st
        self.n = st.ngl
        self.bit = {g: i for i, g in enumerate(st.gluons)}          # gluon particle index -> bit / leaf slot
        # chain nodes: (parent, tree, mask); node 0 = empty prefix
        self.nodes = [(-1, -1, 0)]
        self.node_depth = [0]
        self.closures = []                                           # (prefix node, tree id, key, strings)
        self._walk(tuple(st.gluons), 0, [], colour.Strings({(): 1}))
        keys = sorted({c[2] for c in self.closures})
        self.keys = keys
        self.chan = {k: i for i, k in enumerate(keys)}
        assert len(keys) == st.ndiag, (len(keys), st.ndiag)
        # allowed colour flows per channel: any term with a non-zero coefficient on the flow
        self.allowed = [[0] * len(st.flows) for _ in keys]
        fidx = {f: i for i, f in enumerate(st.flows)}
        for _, _, key, strings in self.closures:
            for word, c in strings.items():
                if c:
                    self.allowed[self.chan[key]][fidx[word]] = 1

    def mask(self, legs):
        m = 0
        for g in legs:
            m |= 1 << self.bit[g]
        return m

    def tree_key(self, tid):
        t = self.st.trees[tid]
        if t.kind == "leaf":
            return str(t.legs[0])
        inner = ",".join(self.tree_key(c) for c in t.children)
        return "(" + inner + ")" if t.kind == "v3" else "[" + inner + "]"

    def _walk(self, remaining, node, blocks, strings):
        st = self.st
        for r in range(1, len(remaining) + 1):
            for blk in itertools.combinations(remaining, r):
                rest = tuple(x for x in remaining if x not in blk)
                for tid in st.trees_on[blk]:
                    s2 = colour.concat(strings, st.trees[tid].strings)
                    if not rest:
                        key = "|".join(self.tree_key(b) for b in blocks + [tid])
                        self.closures.append((node, tid, key, s2))
                    else:
                        self.nodes.append((node, tid, self.nodes[node][2] | self.mask(blk)))
                        self.node_depth.append(self.node_depth[node] + 1)
                        self._walk(rest, len(self.nodes) - 1, blocks + [tid], s2)

    # ------------------------------------------------------------------ tables
    def tree_tasks(self):
        """[(size, words4)] for the non-leaf trees, v3 before v4 within a size."""
        st = self.st
        out = []
        for t in st.trees:
            if t.kind == "leaf":
                continue
            kids = t.children
            a, b = kids[0], kids[1]
            c = kids[2] if t.kind == "v4" else 0
            kind = 0 if t.kind == "v3" else 1
            w0 = t.tid | (kind << 16) | (t.term << 20)
            w1 = a | (b << 16)
            w2 = c | (self.mask(t.legs) << 16)
            w3 = self.mask(st.trees[a].legs) | (self.mask(st.trees[b].legs) << 8)
            out.append((len(t.legs), kind, [w0, w1, w2, w3]))
        out.sort(key=lambda x: (x[0], x[1]))
        return out

    def emit(self):
        st, n, name = self.st, self.n, self.name
        assert len(st.trees) < 65536 and len(self.nodes) < 65536
        for i, g in enumerate(st.gluons):                             # leaves come first, in gluon order
            assert st.trees[i].kind == "leaf" and st.trees[i].legs == (g,)
        tt = self.tree_tasks()
        tree_words, tree_off = [], []
        for size in range(2, n + 1):
            tree_off.append(len(tree_words) // 4)
            for s, _, w in tt:
                if s == size:
                    tree_words += w
        tree_off.append(len(tree_words) // 4)
        chain_words, chain_off = [], []
        maxdepth = max(self.node_depth)
        for d in range(1, maxdepth + 1):
            chain_off.append(len(chain_words) // 2)
            for i, (par, tid, m) in enumerate(self.nodes):
                if self.node_depth[i] == d:
                    chain_words += [i | (par << 16), tid | (m << 16)]
        chain_off.append(len(chain_words) // 2)
        clos_words = []
        for node, tid, key, _ in self.closures:
            clos_words += [node | (tid << 16), self.chan[key]]
        nw = (len(st.flows) + 31) // 32
        flow_words = []
        for row in self.allowed:
            for k in range(4):
                w = 0
                for c in range(32 * k, min(32 * k + 32, len(row))):
                    if row[c]:
                        w |= 1 << (c - 32 * k)
                flow_words.append(w)
        assert nw <= 4
        o = []
        o.append(f"// GENERATED by paper_2503_21935_b200/codegen (emit_diag.py) -- do not edit.  Process {name}:")
        o.append(f"// {st.ndiag} Feynman diagrams = channels, {len(self.closures)} closures (terms), {len(st.trees)} gluon trees, "
                 f"{len(self.nodes)} quark-line prefixes.")
        o.append("#pragma once")
        arr = lambda v: ", ".join(str(x) for x in v)
        o.append(f"__device__ const unsigned int kDiagTree_{name}[] = {{{arr(tree_words)}}};")
        o.append(f"__device__ const unsigned int kDiagChain_{name}[] = {{{arr(chain_words) if chain_words else 0}}};")
        o.append(f"__device__ const unsigned int kDiagClos_{name}[] = {{{arr(clos_words)}}};")
        o.append(f"__device__ const unsigned int kDiagFlows_{name}[] = {{{arr(flow_words)}}};  // [channel][4]: allowed colour flows, bit c")
        o.append(f"struct Diag_{name} {{")
        o.append(f"  static constexpr int n = {n}, npar = {n + 2}, ntree = {len(st.trees)}, nnode = {len(self.nodes)}, "
                 f"nclos = {len(self.closures)}, nchan = {len(self.keys)}, ncol = {len(st.flows)}, nchainlev = {maxdepth};")
        o.append(f"  __device__ __forceinline__ static int tree_off(int i) {{ const int t[] = {{{arr(tree_off)}}}; return t[i]; }}")
        o.append(f"  __device__ __forceinline__ static int chain_off(int i) {{ const int t[] = {{{arr(chain_off)}}}; return t[i]; }}")
        o.append(f"  __device__ __forceinline__ static const unsigned int* tree() {{ return kDiagTree_{name}; }}")
        o.append(f"  __device__ __forceinline__ static const unsigned int* chain() {{ return kDiagChain_{name}; }}")
        o.append(f"  __device__ __forceinline__ static const unsigned int* clos() {{ return kDiagClos_{name}; }}")
        o.append("};")
        return "\n".join(o) + "\n"

    def host_tables(self):
        """C initialisers for me_tables.h: the channel keys (one string, newline separated)."""
        return "\\n".join(self.keys) + "\\n"
