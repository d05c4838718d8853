"""ORACLE, tier 2 (test infrastructure - never imported by the product path): plain block-sparse two-site DMRG.

FP64, numpy only, one small matrix product per block, no batching / fusion / caching.  It follows DESIGN.md C3
(standard complementary-operator QC-DMRG; the paper defers this algorithm to its refs [44, 50, 60], PAPER.md:40,
132, 171, and only fixes WHAT is computed: H of Eq. 1-5, the MPS of Eq. 14, E of Eq. 15, the RDMs of Eq. 9-10).

Formulation: the literal "superblock" one.  For a block X and the neighbouring site s, every operator on the
enlarged block X' = X u {s} is kept as its true matrix on the product basis, as a 4x4 grid of block operators
(EnlargedOp: {(s_out, s_in): BlockOp}).  H_eff at a two-site bond is the bipartition identity between the two
enlarged blocks (L u {i}) and ({i+1} u R):

  H = H_A + H_B + sum_{P in A} (a+_P S_P^B + h.c.) + sum_{P in B} (a+_P S_P^A + h.c.)
      + sum_{P<Q in A} (A_PQ P_PQ^B + h.c.) + sum_{P,S in A} B_PS Q_PS^B                      (C3 step 2)
  S_P^X  = sum_{Q in X} 1/2 t_PQ a_Q + sum_{QRS in X} v_PQRS a+_Q a_R a_S
  P_PQ^X = sum_{RS in X} v_PQRS a_R a_S ,   Q_PS^X = sum_{QR in X} (v_PQRS - v_PQSR) a+_Q a_R  (C3 step 1)

Blocks store the NORMAL operators H, a+_P, A_PQ = a+_P a+_Q (P<Q), B_PS = a+_P a_S and the one-index complementary
S_P; the two-index complementary P, Q are formed from A, B by their definition when needed.  Renormalisation of
an enlarged operator E with the new isometry is X' = sum_{s',s} A[s']^T E[s',s] A[s] (C3 step 3).

Jordan-Wigner convention (C1): spin orbital P = 2p + [dn]; a product written in chain order O_1 O_2 has matrix
elements O_1[a',a] O_2[b',b] (-1)^{parity(O_2) * N(a)} with N(a) the particle number of the INPUT state of part 1.

Pins (tests/test_oracle_dmrg.py): the operator identities against dense Jordan-Wigner matrices; H_eff x against
the tier-1 brute force P^T H P x at every bond; untruncated sweeps against the FCI energy and FCI RDMs; RDM
invariants.  Truncated-D sweep energies are "parity unpinned" beyond variationality (C5).
"""
import numpy as np

SITE_Q = ((0, 0), (1, -1), (1, 1), (2, 0))
SITE_N = (0, 1, 1, 2)


# ----------------------------------------------------------------------------------------------------------------
# Hamiltonian in spin-orbital form
# ----------------------------------------------------------------------------------------------------------------
class Ham:
    """t_PQ = h_pq d(sP,sQ);  v_PQRS = (ps|qr) d(sP,sS) d(sQ,sR);  H = sum t a+a + 1/2 sum v a+a+aa  (C1)."""

    def __init__(self, h, eri):
        self.k = h.shape[0]
        self.h = np.asarray(h, dtype=np.float64)
        self.eri = np.asarray(eri, dtype=np.float64)

    def t(self, P, Q):
        return self.h[P >> 1, Q >> 1] if (P & 1) == (Q & 1) else 0.0

    def v(self, P, Q, R, S):
        if (P & 1) != (S & 1) or (Q & 1) != (R & 1):
            return 0.0
        return self.eri[P >> 1, S >> 1, Q >> 1, R >> 1]

    def w(self, P, Q, R, S):
        return self.v(P, Q, R, S) - self.v(P, Q, S, R)


# site-local annihilators in the basis (|0>, |dn>, |up>, |up dn>), |up dn> = a+_up a+_dn |0>
A_UP = np.zeros((4, 4))
A_UP[0, 2] = 1.0
A_UP[1, 3] = 1.0
A_DN = np.zeros((4, 4))
A_DN[0, 1] = 1.0
A_DN[2, 3] = -1.0


def site_ann(P):
    return A_UP if (P & 1) == 0 else A_DN


def mat_parity(m):
    """Fermion parity (0/1) of a 4x4 site matrix from its non-zero pattern."""
    par = None
    for a in range(4):
        for b in range(4):
            if m[a, b] != 0.0:
                p = (SITE_N[a] - SITE_N[b]) & 1
                assert par is None or par == p
                par = p
    return 0 if par is None else par


# ----------------------------------------------------------------------------------------------------------------
# block operators
# ----------------------------------------------------------------------------------------------------------------
class BlockOp:
    """Operator on a renormalised block basis.  `dq` is the shift of the BOND LABEL (N, 2Sz of everything left of
    the bond): out_label = in_label + dq.  For a left block that is the operator's own quantum-number shift, for a
    right block it is minus that.  blocks: {in_idx: (out_idx, array[d_out, d_in])}."""
    __slots__ = ("dq", "par", "blocks")

    def __init__(self, dq, par, blocks=None):
        self.dq, self.par, self.blocks = (int(dq[0]), int(dq[1])), int(par), ({} if blocks is None else blocks)

    def T(self):
        return BlockOp((-self.dq[0], -self.dq[1]), self.par,
                       {o: (i, np.ascontiguousarray(a.T)) for i, (o, a) in self.blocks.items()})

    def scaled(self, c):
        return BlockOp(self.dq, self.par, {i: (o, c * a) for i, (o, a) in self.blocks.items()})

    def add(self, c, other):
        assert self.dq == other.dq and self.par == other.par
        for i, (o, a) in other.blocks.items():
            if i in self.blocks:
                self.blocks[i] = (o, self.blocks[i][1] + c * a)
            else:
                self.blocks[i] = (o, c * a)

    def nnz(self):
        return sum(a.size for _, a in self.blocks.values())


def identity_op(basis):
    return BlockOp((0, 0), 0, {i: (i, np.eye(d)) for i, (_, _, d) in enumerate(basis)})


class EnlargedOp:
    """True matrix of an operator on (block x site) or (site x block): {(s_out, s_in): BlockOp}."""
    __slots__ = ("dq", "par", "grid")

    def __init__(self, dq, par):
        self.dq, self.par, self.grid = (int(dq[0]), int(dq[1])), int(par), {}

    def T(self):
        e = EnlargedOp((-self.dq[0], -self.dq[1]), self.par)
        e.grid = {(si, so): op.T() for (so, si), op in self.grid.items()}
        return e

    def add(self, c, other):
        assert self.dq == other.dq and self.par == other.par
        for key, op in other.grid.items():
            if key in self.grid:
                self.grid[key].add(c, op)
            else:
                self.grid[key] = op.scaled(c)


class Block:
    """A renormalised block: side 'L' (sites [0,b)) or 'R' (sites [b,k)), its bond basis, and its operators
    ops[key] with keys ('H',), ('C',P), ('S',P), ('A',P,Q) P<Q, ('B',P,S)."""

    def __init__(self, side, b, k, basis):
        self.side, self.b, self.k = side, b, k
        self.basis = basis
        self.index = {(n, s): i for i, (n, s, d) in enumerate(basis)}
        self.ops = {}
        self.eye = identity_op(basis)

    def inside(self):
        return list(range(0, 2 * self.b)) if self.side == "L" else list(range(2 * self.b, 2 * self.k))

    def sgn(self):
        """+1: label shift = operator shift (left block);  -1 for a right block."""
        return 1 if self.side == "L" else -1


def empty_block(side, k, mps):
    b = 0 if side == "L" else k
    blk = Block(side, b, k, mps["bonds"][b])
    blk.ops[("H",)] = BlockOp((0, 0), 0, {0: (0, np.zeros((1, 1)))})
    for P in range(2 * k):                                   # S_P of the empty block is the zero operator
        g = blk.sgn()
        blk.ops[("S", P)] = BlockOp((-g, -g * (1 if (P & 1) == 0 else -1)), 1)
    return blk


# ----------------------------------------------------------------------------------------------------------------
# complementary two-index operators of a block from its normal operators, by definition (C3 step 1)
# ----------------------------------------------------------------------------------------------------------------
def _stacked(blk, kind):
    """All stored operators of one kind on a block, grouped by label shift and laid side by side per in-sector:
    {dq: (keys, {in_idx: (out_idx, array[n_ops, d_out, d_in], present[n_ops])})}.  Built once per block (its operators
    never change after construction).  Only a container: it lets the defining sums of compl_P / compl_Q below run as
    one library contraction (np.tensordot over the operator index) instead of a Python loop of block additions."""
    cache = blk.__dict__.setdefault("_stacks", {})
    if kind not in cache:
        groups = {}
        for key, op in blk.ops.items():
            if key[0] == kind:
                groups.setdefault(op.dq, []).append(key)
        out = {}
        for dq, keys in groups.items():
            arrs = {}
            for i in sorted({i for key in keys for i in blk.ops[key].blocks}):
                first = next(blk.ops[key].blocks[i] for key in keys if i in blk.ops[key].blocks)
                st = np.zeros((len(keys),) + first[1].shape)
                present = np.zeros(len(keys), dtype=bool)
                for n, key in enumerate(keys):
                    if i in blk.ops[key].blocks:
                        assert blk.ops[key].blocks[i][0] == first[0]
                        st[n] = blk.ops[key].blocks[i][1]
                        present[n] = True
                arrs[i] = (first[0], st, present)
            out[dq] = (keys, arrs)
        cache[kind] = out
    return cache[kind]


def compl_P(blk, ham, P, Q):
    """P_PQ^X = sum_{R,S in X} v_PQRS a_R a_S = sum_{R<S in X} (v_PQSR - v_PQRS) (A_RS)^T  (C3 step 1); the sum over
    the stored A_RS (those whose shift matches) is one tensordot per block."""
    g = blk.sgn()
    dq = (-2, -((1 if P % 2 == 0 else -1) + (1 if Q % 2 == 0 else -1)))
    out = BlockOp((g * dq[0], g * dq[1]), 0)
    entry = _stacked(blk, "A").get((-out.dq[0], -out.dq[1]))          # A_RS carries the opposite label shift
    if entry is None:
        return out
    keys, arrs = entry
    c = np.array([ham.v(P, Q, S, R) - ham.v(P, Q, R, S) for (_, R, S) in keys])
    nz = c != 0.0
    for i, (o, st, present) in arrs.items():
        if np.any(nz & present):
            out.blocks[o] = (i, np.ascontiguousarray(np.tensordot(c, st, axes=1).T))
    return out


def compl_Q(blk, ham, P, S):
    """Q_PS^X = sum_{Q,R in X} (v_PQRS - v_PQSR) a+_Q a_R  (C3 step 1); one tensordot over the stored B_QR per block."""
    g = blk.sgn()
    dq = (0, -(1 if P % 2 == 0 else -1) + (1 if S % 2 == 0 else -1))
    out = BlockOp((g * dq[0], g * dq[1]), 0)
    entry = _stacked(blk, "B").get(out.dq)
    if entry is None:
        return out
    keys, arrs = entry
    c = np.array([ham.w(P, Q, R, S) for (_, Q, R) in keys])
    nz = c != 0.0
    for i, (o, st, present) in arrs.items():
        if np.any(nz & present):
            out.blocks[i] = (o, np.tensordot(c, st, axes=1))
    return out


# ----------------------------------------------------------------------------------------------------------------
# enlarged-block operators (block x site for a left block, site x block for a right block)
# ----------------------------------------------------------------------------------------------------------------
def spin_of(P):
    return 1 if (P & 1) == 0 else -1


class Enlarger:
    """Operators of X' = X u {site p} as EnlargedOps.  Left block: p = b (site after the block);
    right block: p = b-1 (site before the block)."""

    def __init__(self, blk, ham, p):
        assert p == (blk.b if blk.side == "L" else blk.b - 1)
        self.blk, self.ham, self.p = blk, ham, p
        self.site = [2 * p, 2 * p + 1]
        self.X = blk.inside()
        self.g = blk.sgn()
        self._pc, self._qc = {}, {}

    # -- helpers ----------------------------------------------------------------------------------------------
    def new(self, shift, par):
        return EnlargedOp((self.g * shift[0], self.g * shift[1]), par)

    def piece(self, E, coef, O, m, written="bs"):
        """Add coef * (O . m) ('bs': block op written first) or coef * (m . O) ('sb') to E, as true matrix
        elements on the product basis in chain order (Jordan-Wigner rule of C1)."""
        if O is None:
            O = self.blk.eye
        pm, po = mat_parity(m), O.par
        assert (pm ^ po) == E.par
        chain = "bs" if self.blk.side == "L" else "sb"
        if written != chain and pm == 1 and po == 1:
            coef = -coef
        for so in range(4):
            for si in range(4):
                if m[so, si] == 0.0:
                    continue
                dqs = (SITE_Q[so][0] - SITE_Q[si][0], SITE_Q[so][1] - SITE_Q[si][1])
                if self.blk.side == "L":
                    assert (O.dq[0] + dqs[0], O.dq[1] + dqs[1]) == E.dq
                    blocks = {}
                    for i, (o, a) in O.blocks.items():
                        sgn = -1.0 if (pm and (self.blk.basis[i][0] & 1)) else 1.0
                        blocks[i] = (o, (coef * m[so, si] * sgn) * a)
                    op = BlockOp(O.dq, O.par, blocks)
                else:
                    assert (O.dq[0] - dqs[0], O.dq[1] - dqs[1]) == E.dq
                    sgn = -1.0 if (po and (SITE_N[si] & 1)) else 1.0
                    op = O.scaled(coef * m[so, si] * sgn)
                if (so, si) in E.grid:
                    E.grid[(so, si)].add(1.0, op)
                else:
                    E.grid[(so, si)] = op

    def Pc_blk(self, P, Q):
        if (P, Q) not in self._pc:
            self._pc[(P, Q)] = compl_P(self.blk, self.ham, P, Q)
        return self._pc[(P, Q)]

    def Qc_blk(self, P, S):
        if (P, S) not in self._qc:
            self._qc[(P, S)] = compl_Q(self.blk, self.ham, P, S)
        return self._qc[(P, S)]

    # site-local 4x4 matrices by definition
    def s_H(self):
        h, m = self.ham, np.zeros((4, 4))
        for P in self.site:
            for Q in self.site:
                m += h.t(P, Q) * site_ann(P).T @ site_ann(Q)
                for R in self.site:
                    for S in self.site:
                        m += 0.5 * h.v(P, Q, R, S) * site_ann(P).T @ site_ann(Q).T @ site_ann(R) @ site_ann(S)
        return m

    def s_S(self, P):
        h, m = self.ham, np.zeros((4, 4))
        for Q in self.site:
            m += 0.5 * h.t(P, Q) * site_ann(Q)
            for R in self.site:
                for S in self.site:
                    m += h.v(P, Q, R, S) * site_ann(Q).T @ site_ann(R) @ site_ann(S)
        return m

    def s_P(self, P, Q):
        m = np.zeros((4, 4))
        for R in self.site:
            for S in self.site:
                m += self.ham.v(P, Q, R, S) * site_ann(R) @ site_ann(S)
        return m

    def s_Q(self, P, S):
        m = np.zeros((4, 4))
        for Q in self.site:
            for R in self.site:
                m += self.ham.w(P, Q, R, S) * site_ann(Q).T @ site_ann(R)
        return m

    # -- enlarged operators -----------------------------------------------------------------------------------
    def ident(self):
        E = self.new((0, 0), 0)
        self.piece(E, 1.0, None, np.eye(4))
        return E

    def H(self):
        ops = self.blk.ops
        E = self.new((0, 0), 0)
        self.piece(E, 1.0, ops[("H",)], np.eye(4))
        self.piece(E, 1.0, None, self.s_H())
        G = self.new((0, 0), 0)
        for P in self.X:                                                   # a+_P^X S_P^s
            self.piece(G, 1.0, ops[("C", P)], self.s_S(P), "bs")
        for P in self.site:                                                # a+_P^s S_P^X
            self.piece(G, 1.0, ops[("S", P)], site_ann(P).T, "sb")
        P, Q = self.site                                                   # A^s_PQ P^X_PQ (P<Q in the site)
        if self.X:
            self.piece(G, 1.0, self.Pc_blk(P, Q), site_ann(P).T @ site_ann(Q).T, "sb")
        E.add(1.0, G)
        E.add(1.0, G.T())
        if self.X:
            for P in self.site:                                            # B^s_PS Q^X_PS
                for S in self.site:
                    self.piece(E, 1.0, self.Qc_blk(P, S), site_ann(P).T @ site_ann(S), "sb")
        return E

    def C(self, P):
        E = self.new((1, spin_of(P)), 1)
        if P in self.site:
            self.piece(E, 1.0, None, site_ann(P).T)
        else:
            self.piece(E, 1.0, self.blk.ops[("C", P)], np.eye(4))
        return E

    def A(self, P, Q):
        """a+_P a+_Q, P < Q, both inside X'."""
        assert P < Q
        E = self.new((2, spin_of(P) + spin_of(Q)), 0)
        ps, qs = P in self.site, Q in self.site
        if ps and qs:
            self.piece(E, 1.0, None, site_ann(P).T @ site_ann(Q).T)
        elif not ps and not qs:
            self.piece(E, 1.0, self.blk.ops[("A", P, Q)], np.eye(4))
        elif qs:                                                           # a+_P^X a+_Q^s
            self.piece(E, 1.0, self.blk.ops[("C", P)], site_ann(Q).T, "bs")
        else:                                                              # a+_P^s a+_Q^X
            self.piece(E, 1.0, self.blk.ops[("C", Q)], site_ann(P).T, "sb")
        return E

    def B(self, P, S):
        """a+_P a_S, both inside X'."""
        E = self.new((0, spin_of(P) - spin_of(S)), 0)
        ps, ss = P in self.site, S in self.site
        if ps and ss:
            self.piece(E, 1.0, None, site_ann(P).T @ site_ann(S))
        elif not ps and not ss:
            self.piece(E, 1.0, self.blk.ops[("B", P, S)], np.eye(4))
        elif ss:                                                           # a+_P^X a_S^s
            self.piece(E, 1.0, self.blk.ops[("C", P)], site_ann(S), "bs")
        else:                                                              # a+_P^s a_S^X
            self.piece(E, 1.0, self.blk.ops[("C", S)].T(), site_ann(P).T, "sb")
        return E

    def S(self, P):
        """S_P^{X'} for P outside X' (C3 step 3, first recurrence)."""
        ops = self.blk.ops
        E = self.new((-1, -spin_of(P)), 1)
        self.piece(E, 1.0, ops[("S", P)], np.eye(4))
        self.piece(E, 1.0, None, self.s_S(P))
        for Q in self.X:                                                   # a+_Q^X P^s_PQ
            m = self.s_P(P, Q)
            if np.any(m):
                self.piece(E, 1.0, ops[("C", Q)], m, "bs")
        for S in self.X:                                                   # Q^s_PS a_S^X
            m = self.s_Q(P, S)
            if np.any(m):
                self.piece(E, 1.0, ops[("C", S)].T(), m, "sb")
        if self.X:
            for Q in self.site:                                            # a+_Q^s P^X_PQ
                self.piece(E, 1.0, self.Pc_blk(P, Q), site_ann(Q).T, "sb")
            for S in self.site:                                            # Q^X_PS a_S^s
                self.piece(E, 1.0, self.Qc_blk(P, S), site_ann(S), "bs")
        return E

    def Pc(self, P, Q):
        """P_PQ^{X'} for P, Q outside X' (second recurrence)."""
        E = self.new((-2, -(spin_of(P) + spin_of(Q))), 0)
        if self.X:
            self.piece(E, 1.0, self.Pc_blk(P, Q), np.eye(4))
        m = self.s_P(P, Q)
        if np.any(m):
            self.piece(E, 1.0, None, m)
        for R in self.X:
            for S in self.site:                                            # (v_PQRS - v_PQSR) a_R^X a_S^s
                c = self.ham.w(P, Q, R, S)
                if c != 0.0:
                    self.piece(E, c, self.blk.ops[("C", R)].T(), site_ann(S), "bs")
        return E

    def Qc(self, P, S):
        """Q_PS^{X'} for P, S outside X' (third recurrence)."""
        E = self.new((0, -spin_of(P) + spin_of(S)), 0)
        if self.X:
            self.piece(E, 1.0, self.Qc_blk(P, S), np.eye(4))
        m = self.s_Q(P, S)
        if np.any(m):
            self.piece(E, 1.0, None, m)
        for Q in self.X:
            for R in self.site:                                            # w_PQRS a+_Q^X a_R^s
                c = self.ham.w(P, Q, R, S)
                if c != 0.0:
                    self.piece(E, c, self.blk.ops[("C", Q)], site_ann(R), "bs")
        for Q in self.site:
            for R in self.X:                                               # w_PQRS a+_Q^s a_R^X
                c = self.ham.w(P, Q, R, S)
                if c != 0.0:
                    self.piece(E, c, self.blk.ops[("C", R)].T(), site_ann(Q).T, "sb")
        return E


# ----------------------------------------------------------------------------------------------------------------
# renormalisation (blocking): X' = sum_{s',s} A[s']^T E[s',s] A[s]   (left)   /   B[s'] E[s',s] B[s]^T   (right)
# ----------------------------------------------------------------------------------------------------------------
def rotate(E, blk, tensor, new_basis):
    nidx = {(n, s): i for i, (n, s, d) in enumerate(new_basis)}
    out = BlockOp(E.dq, E.par)
    for (so, si), op in E.grid.items():
        for i, (o, a) in op.blocks.items():
            if blk.side == "L":
                ti, to = tensor.get((i, si)), tensor.get((o, so))
                if ti is None or to is None:
                    continue
                n, s, _ = blk.basis[i]
                ni = nidx[(n + SITE_Q[si][0], s + SITE_Q[si][1])]
                n, s, _ = blk.basis[o]
                no = nidx[(n + SITE_Q[so][0], s + SITE_Q[so][1])]
                val = to.T @ a @ ti
            else:
                n, s, _ = blk.basis[i]
                key_i = (n - SITE_Q[si][0], s - SITE_Q[si][1])
                n, s, _ = blk.basis[o]
                key_o = (n - SITE_Q[so][0], s - SITE_Q[so][1])
                if key_i not in nidx or key_o not in nidx:
                    continue
                ni, no = nidx[key_i], nidx[key_o]
                ti, to = tensor.get((ni, si)), tensor.get((no, so))
                if ti is None or to is None:
                    continue
                val = to @ a @ ti.T
            if ni in out.blocks:
                out.blocks[ni] = (no, out.blocks[ni][1] + val)
            else:
                out.blocks[ni] = (no, val)
    return out


def grow(blk, ham, mps_bonds, tensor):
    """One blocking step: L_b -> L_{b+1} with the left-orthonormal tensor of site b, or R_b -> R_{b-1} with the
    right-orthonormal tensor of site b-1.  Keeps H, a+_P, A_PQ, B_PS (inside) and S_P (outside)."""
    k = blk.k
    if blk.side == "L":
        p, nb = blk.b, blk.b + 1
    else:
        p, nb = blk.b - 1, blk.b - 1
    en = Enlarger(blk, ham, p)
    new = Block(blk.side, nb, k, mps_bonds[nb])
    inside = new.inside()
    outside = [P for P in range(2 * k) if P not in set(inside)]
    rot = lambda E: rotate(E, blk, tensor, new.basis)
    new.ops[("H",)] = rot(en.H())
    for P in inside:
        new.ops[("C", P)] = rot(en.C(P))
    for a_, P in enumerate(inside):
        for Q in inside[a_ + 1:]:
            new.ops[("A", P, Q)] = rot(en.A(P, Q))
        for S in inside:
            new.ops[("B", P, S)] = rot(en.B(P, S))
    for P in outside:
        new.ops[("S", P)] = rot(en.S(P))
    return new


# ----------------------------------------------------------------------------------------------------------------
# H_eff x at a two-site bond (C3 step 5)
# ----------------------------------------------------------------------------------------------------------------
def psi_layout(bonds_l, bonds_r, target):
    """Blocks (l_idx, s_i, s_j, r_idx, rows, cols, offset) ordered by (l_idx, s_i, s_j)."""
    rindex = {(n, s): j for j, (n, s, d) in enumerate(bonds_r)}
    out, off = [], 0
    for li, (n, s, dl) in enumerate(bonds_l):
        for a in range(4):
            for b in range(4):
                key = (n + SITE_Q[a][0] + SITE_Q[b][0], s + SITE_Q[a][1] + SITE_Q[b][1])
                if key in rindex:
                    ri = rindex[key]
                    out.append((li, a, b, ri, dl, bonds_r[ri][2], off))
                    off += dl * bonds_r[ri][2]
    return out, off


def flat_to_blocks(layout, x):
    return {(li, a, b): x[off:off + m * n].reshape(m, n) for (li, a, b, ri, m, n, off) in layout}


def blocks_to_flat(layout, nnz, blocks):
    y = np.zeros(nnz)
    for (li, a, b, ri, m, n, off) in layout:
        if (li, a, b) in blocks:
            y[off:off + m * n] = blocks[(li, a, b)].ravel()
    return y


class Heff:
    """H_eff at two-site bond i from a left block L_i and a right block R_{i+2}."""

    def __init__(self, LB, RB, ham, i, normal_side=None):
        k = ham.k
        assert LB.side == "L" and LB.b == i and RB.side == "R" and RB.b == i + 2
        self.LB, self.RB, self.i, self.k = LB, RB, i, k
        self.layout, self.nnz = psi_layout(LB.basis, RB.basis, None)
        self.by_key = {(li, a, b): (ri, m, n) for (li, a, b, ri, m, n, off) in self.layout}
        if normal_side is None:
            normal_side = "L" if (i + 1) <= (k - i - 1) else "R"
        self.normal_side = normal_side
        el, er = Enlarger(LB, ham, i), Enlarger(RB, ham, i + 1)
        A = list(range(0, 2 * i + 2))
        B = list(range(2 * i + 2, 2 * k))
        T = []                                         # (coef, E on L u i, F on j u R, add_hc)
        T.append((1.0, el.H(), er.ident(), False))
        T.append((1.0, el.ident(), er.H(), False))
        for P in A:                                    # a+_P^A S_P^B + h.c.
            T.append((1.0, el.C(P), er.S(P), True))
        for P in B:                                    # a+_P^B S_P^A = - S_P^A a+_P^B
            T.append((-1.0, el.S(P), er.C(P), True))
        if normal_side == "L":
            for a_, P in enumerate(A):
                for Q in A[a_ + 1:]:
                    T.append((1.0, el.A(P, Q), er.Pc(P, Q), True))
                for S in A:
                    T.append((1.0, el.B(P, S), er.Qc(P, S), False))
        else:
            for a_, P in enumerate(B):
                for Q in B[a_ + 1:]:
                    T.append((1.0, el.Pc(P, Q), er.A(P, Q), True))
                for S in B:
                    T.append((1.0, el.Qc(P, S), er.B(P, S), False))
        self.terms = T

    def apply_blocks(self, xb):
        yb = {key: np.zeros((m, n)) for key, (ri, m, n) in self.by_key.items()}
        LBs = self.LB.basis
        for (coef, E, F, hc) in self.terms:
            for (ao, ai), OL in E.grid.items():
                for (bo, bi), OR in F.grid.items():
                    for li, (lo, ml) in OL.blocks.items():
                        kin = (li, ai, bi)
                        if kin not in self.by_key:
                            continue
                        ri = self.by_key[kin][0]
                        if ri not in OR.blocks:
                            continue
                        ro, mr = OR.blocks[ri]
                        kout = (lo, ao, bo)
                        if kout not in self.by_key:
                            continue
                        assert self.by_key[kout][0] == ro
                        sgn = -1.0 if (F.par and ((LBs[li][0] + SITE_N[ai]) & 1)) else 1.0
                        c = coef * sgn
                        yb[kout] += c * (ml @ xb[kin] @ mr.T)
                        if hc:
                            yb[kin] += c * (ml.T @ xb[kout] @ mr)
        return yb

    def apply(self, x):
        return blocks_to_flat(self.layout, self.nnz, self.apply_blocks(flat_to_blocks(self.layout, x)))

    def gemm_flops(self):
        """Flops of the matrix products one apply() executes, counted by walking the term list with the loop
        structure of apply_blocks: (ml @ x) @ mr^T = 2 d_lo d_li d_ri + 2 d_lo d_ri d_ro per (term, site-state pair,
        block), and the same again with the transposed factors for terms that add their Hermitian conjugate.
        Integer bookkeeping only - no arithmetic of the method is done here."""
        f = 0
        for (coef, E, F, hc) in self.terms:
            for (ao, ai), OL in E.grid.items():
                for (bo, bi), OR in F.grid.items():
                    for li, (lo, ml) in OL.blocks.items():
                        kin = (li, ai, bi)
                        if kin not in self.by_key:
                            continue
                        ri, m_in, n_in = self.by_key[kin]
                        if ri not in OR.blocks or (lo, ao, bo) not in self.by_key:
                            continue
                        m_out, n_out = ml.shape[0], OR.blocks[ri][1].shape[0]
                        f += 2 * m_out * m_in * n_in + 2 * m_out * n_in * n_out
                        if hc:
                            f += 2 * m_in * m_out * n_out + 2 * m_in * n_out * n_in
        return float(f)

    def diagonal(self):
        """diag(H_eff) for the Davidson preconditioner: terms with all four factors on the diagonal."""
        db = {key: np.zeros((m, n)) for key, (ri, m, n) in self.by_key.items()}
        LBs = self.LB.basis
        for (coef, E, F, hc) in self.terms:
            for (ao, ai), OL in E.grid.items():
                if ao != ai:
                    continue
                for (bo, bi), OR in F.grid.items():
                    if bo != bi:
                        continue
                    for li, (lo, ml) in OL.blocks.items():
                        if lo != li or (li, ai, bi) not in self.by_key:
                            continue
                        ri = self.by_key[(li, ai, bi)][0]
                        if ri not in OR.blocks or OR.blocks[ri][0] != ri:
                            continue
                        sgn = -1.0 if (F.par and ((LBs[li][0] + SITE_N[ai]) & 1)) else 1.0
                        c = coef * sgn * (2.0 if hc else 1.0)
                        db[(li, ai, bi)] += c * np.outer(np.diag(ml), np.diag(OR.blocks[ri][1]))
        return blocks_to_flat(self.layout, self.nnz, db)


def build_left(mps, ham, upto):
    """Left blocks L_0 .. L_upto from the (left-orthonormal) tensors of sites < upto."""
    blocks = [empty_block("L", ham.k, mps)]
    for p in range(upto):
        blocks.append(grow(blocks[-1], ham, mps["bonds"], mps["tensors"][p]))
    return blocks


def build_right(mps, ham, downto):
    """Right blocks R_k .. R_downto (returned indexed by bond: dict) from the tensors of sites >= downto."""
    k = ham.k
    blocks = {k: empty_block("R", k, mps)}
    for b in range(k, downto, -1):
        blocks[b - 1] = grow(blocks[b], ham, mps["bonds"], mps["tensors"][b - 1])
    return blocks


# ----------------------------------------------------------------------------------------------------------------
# Davidson (reading S13): single root, diagonal preconditioner, double Gram-Schmidt, restart
# ----------------------------------------------------------------------------------------------------------------
def davidson(apply, diag, x0, tol=1e-7, max_iter=100, max_subspace=20):
    """Lowest eigenpair of the symmetric operator `apply`.  Returns (theta, u, n_matvec, residual_norm, ok)."""
    v = x0 / np.linalg.norm(x0)
    V, W = [v], [apply(v)]
    nmv = 1
    theta, u, rn = 0.0, v, np.inf
    for _ in range(max_iter):
        m = len(V)
        Vm, Wm = np.array(V), np.array(W)
        Hs = Vm @ Wm.T
        Hs = 0.5 * (Hs + Hs.T)
        ev, es = np.linalg.eigh(Hs)
        theta, s = ev[0], es[:, 0]
        u = s @ Vm
        hu = s @ Wm
        r = hu - theta * u
        rn = np.linalg.norm(r)
        if rn <= tol:
            return theta, u / np.linalg.norm(u), nmv, rn, True
        den = diag - theta
        small = np.abs(den) < 1e-8
        den = np.where(small, np.where(den < 0, -1e-8, 1e-8), den)
        t = r / den
        if m >= max_subspace:
            nu = np.linalg.norm(u)
            V, W = [u / nu], [hu / nu]
        for _gs in range(2):
            for vv in V:
                t = t - (vv @ t) * vv
        nt = np.linalg.norm(t)
        if nt < 1e-14:
            break
        t = t / nt
        V.append(t)
        W.append(apply(t))
        nmv += 1
    return theta, u / np.linalg.norm(u), nmv, rn, False


def lanczos(apply, x0, tol=1e-7, max_iter=100, max_subspace=20):
    """Lowest eigenpair of the symmetric operator `apply` by the Lanczos method, the paper's other local eigensolver
    ("Lanczos and Davidson diagonalization methods"; reading S33): Krylov vectors
    v_{j+1} beta_{j+1} = H v_j - alpha_j v_j - beta_j v_{j-1}, re-orthogonalised against all stored vectors (twice),
    Rayleigh-Ritz on the tridiagonal matrix, residual norm beta_{j+1} |s_j|, restart from the Ritz vector when
    max_subspace vectors are stored.  Returns (theta, u, n_matvec, residual_norm, ok) like davidson()."""
    v = x0 / np.linalg.norm(x0)
    V, alphas, betas = [v], [], []
    nmv = 0
    theta, u, rn = 0.0, v, np.inf
    for _ in range(max_iter):
        w = apply(V[-1])
        nmv += 1
        alphas.append(float(V[-1] @ w))
        w = w - alphas[-1] * V[-1]
        if len(V) > 1:
            w = w - betas[-1] * V[-2]
        for _gs in range(2):
            for vv in V:
                w = w - (vv @ w) * vv
        beta = float(np.linalg.norm(w))
        m = len(V)
        T = np.diag(alphas) + np.diag(betas, 1) + np.diag(betas, -1)
        ev, es = np.linalg.eigh(T)
        theta, s = ev[0], es[:, 0]
        u = s @ np.array(V)
        rn = abs(beta * s[-1])
        if rn <= tol:
            return theta, u / np.linalg.norm(u), nmv, rn, True
        if beta < 1e-14:
            break
        if m >= max_subspace:
            V, alphas, betas = [u / np.linalg.norm(u)], [], []
            continue
        betas.append(beta)
        V.append(w / beta)
    return theta, u / np.linalg.norm(u), nmv, rn, False


def sweeps_converged(energies, eps_sweep):
    """Stopping rule of the sweep loop ("terminated when the energy difference between three subsequent
    sweeps falls below ... eps_sweep"; reading S34): true once the last three sweep energies E_{s-2}, E_{s-1}, E_s
    differ pairwise-consecutively by less than eps_sweep."""
    if len(energies) < 3:
        return False
    a, b, c = energies[-3:]
    return abs(b - a) < eps_sweep and abs(c - b) < eps_sweep


# ----------------------------------------------------------------------------------------------------------------
# decomposition and truncation (reading S14) and the two-site sweep (readings S12, S16-S18)
# ----------------------------------------------------------------------------------------------------------------
def select_kept(sv_sorted, D, sv_floor=1e-10, cluster_rel_gap=1e-6, dbss_eps=0.0, dbss_dmin=0):
    """Number of kept states from the pooled singular values of the normalised two-site state, sorted descending.
    Fixed D (reading S14): m = min(D, #sigma > floor); while the cut falls inside a near-degenerate cluster
    (sigma_{m+1} >= (1 - gap) sigma_m) decrease m; if that empties the bond keep the original m.
    DBSS (fixed truncation error eps_TR with a minimal bond dimension D_min; reading S32):
    m_eps = the fewest states whose discarded weight 1 - sum_{t < m} sigma_t^2 is <= eps_TR, then
    m = min(max(m_eps, D_min), D_max = D, #sigma > floor); a cut inside a cluster is moved UP to the end of the
    cluster when that stays within min(D_max, count) (the error target stays met), otherwise down as in S14."""
    count = sum(1 for sv in sv_sorted if sv > sv_floor)
    cap = min(D, count)
    inside = lambda m: 0 < m < count and sv_sorted[m] >= (1.0 - cluster_rel_gap) * sv_sorted[m - 1]
    if dbss_eps > 0.0:
        kept_w, m = 0.0, 0
        while m < count and 1.0 - kept_w > dbss_eps:
            kept_w += sv_sorted[m] ** 2
            m += 1
        m = min(max(m, dbss_dmin), cap)
        up = m
        while inside(up):
            up += 1
        if up <= cap:
            return up
    else:
        m = cap
    m0 = m
    while inside(m):
        m -= 1
    return m0 if m == 0 else m


def split_theta(theta_blocks, bonds_l, bonds_r, D, direction, sv_floor=1e-10, cluster_rel_gap=1e-6, dbss_eps=0.0,
                dbss_dmin=0):
    """SVD of the two-site tensor per enlarged-left sector, global selection of the kept states by select_kept (fixed
    D or DBSS; never cuts through a near-degenerate cluster).  Returns (mid_basis, A blocks {(l,a): [d_l,d_m]},
    B blocks {(m,b): [d_m,d_r]}, trunc_err, kept) with singular values absorbed to the right ('fwd') or to the left
    ('bwd')."""
    rindex = {(n, s): j for j, (n, s, d) in enumerate(bonds_r)}
    sectors = {}
    for (li, a, b), blk in theta_blocks.items():
        n, s, _ = bonds_l[li]
        q = (n + SITE_Q[a][0], s + SITE_Q[a][1])
        sec = sectors.setdefault(q, dict(rows=set(), cols=set()))
        ri = rindex[(q[0] + SITE_Q[b][0], q[1] + SITE_Q[b][1])]
        sec["rows"].add((li, a))
        sec["cols"].add((b, ri))
    nrm = np.sqrt(sum(np.sum(v * v) for v in theta_blocks.values()))
    svds = {}
    pool = []
    for q in sorted(sectors.keys()):
        rows, cols = sorted(sectors[q]["rows"]), sorted(sectors[q]["cols"])
        roff, coff = {}, {}
        o = 0
        for (li, a) in rows:
            roff[(li, a)] = o
            o += bonds_l[li][2]
        nr = o
        o = 0
        for (b, ri) in cols:
            coff[(b, ri)] = o
            o += bonds_r[ri][2]
        nc = o
        M = np.zeros((nr, nc))
        for (li, a) in rows:
            for (b, ri) in cols:
                blk = theta_blocks.get((li, a, b))
                if blk is not None and rindex.get((q[0] + SITE_Q[b][0], q[1] + SITE_Q[b][1])) == ri:
                    M[roff[(li, a)]:roff[(li, a)] + blk.shape[0], coff[(b, ri)]:coff[(b, ri)] + blk.shape[1]] = blk
        U, S, Vt = np.linalg.svd(M / nrm, full_matrices=False)
        svds[q] = (rows, cols, roff, coff, U, S, Vt)
        for j, sv in enumerate(S):
            pool.append((sv, q, j))
    order = sorted(range(len(pool)), key=lambda t: -pool[t][0])       # stable: ties by (sector, index)
    sv_sorted = [pool[t][0] for t in order]
    m = select_kept(sv_sorted, D, sv_floor, cluster_rel_gap, dbss_eps, dbss_dmin)
    keep = {}
    for t in order[:m]:
        _, q, j = pool[t]
        keep.setdefault(q, []).append(j)
    kept_w = sum(sv_sorted[t] ** 2 for t in range(m))
    trunc = max(0.0, 1.0 - kept_w)
    scale = 1.0 / np.sqrt(kept_w)
    mid_basis = [(q[0], q[1], len(keep[q])) for q in sorted(keep.keys())]
    Ab, Bb = {}, {}
    for mi, (n, s, dm) in enumerate(mid_basis):
        rows, cols, roff, coff, U, S, Vt = svds[(n, s)]
        js = sorted(keep[(n, s)])
        Uk, Sk, Vk = U[:, js], S[js] * scale, Vt[js, :]
        if direction == "fwd":
            Vk = Sk[:, None] * Vk
        else:
            Uk = Uk * Sk[None, :]
        for (li, a) in rows:
            Ab[(li, a)] = np.ascontiguousarray(Uk[roff[(li, a)]:roff[(li, a)] + bonds_l[li][2], :])
        for (b, ri) in cols:
            Bb[(mi, b)] = np.ascontiguousarray(Vk[:, coff[(b, ri)]:coff[(b, ri)] + bonds_r[ri][2]])
    return mid_basis, Ab, Bb, trunc, m


def two_site_tensor(mps, i):
    """theta[l, a, b, r] = sum_m T_i[(l,a)][:, m] T_{i+1}[(m,b)][m, :] as psi-layout blocks."""
    mid = {(n, s): j for j, (n, s, d) in enumerate(mps["bonds"][i + 1])}
    out = {}
    for (li, a), ta in mps["tensors"][i].items():
        n, s, _ = mps["bonds"][i][li]
        mi = mid[(n + SITE_Q[a][0], s + SITE_Q[a][1])]
        for b in range(4):
            tb = mps["tensors"][i + 1].get((mi, b))
            if tb is not None:
                out[(li, a, b)] = ta @ tb
    return out


class SweepEngine:
    """Two-site fixed-D DMRG on an imported right-canonical MPS (C3 step 4).  One call of sweep() = forward pass
    over bonds 0..k-2 then backward pass k-2..0 (reading S12)."""

    def __init__(self, h, eri, mps, davidson_tol=1e-7, davidson_max_iter=100, davidson_max_subspace=20, dbss_eps=0.0,
                 dbss_dmin=0, eigensolver="davidson"):
        self.ham = Ham(h, eri)
        self.k = self.ham.k
        self.mps = dict(mps)
        self.mps["bonds"] = [list(b) for b in mps["bonds"]]
        self.mps["tensors"] = [dict(t) for t in mps["tensors"]]
        self.mps["gauge"] = list(mps["gauge"])
        self.opts = dict(tol=davidson_tol, max_iter=davidson_max_iter, max_subspace=davidson_max_subspace)
        self.dbss = dict(dbss_eps=dbss_eps, dbss_dmin=dbss_dmin)
        self.eigensolver = eigensolver
        self.L = {0: empty_block("L", self.k, self.mps)}
        self.R = build_right(self.mps, self.ham, 2)
        self.log = []

    def _optimise(self, i, D, direction):
        mps, ham = self.mps, self.ham
        H = Heff(self.L[i], self.R[i + 2], ham, i)
        guess = blocks_to_flat(H.layout, H.nnz, two_site_tensor(mps, i))
        if self.eigensolver == "lanczos":
            theta, u, nmv, rn, ok = lanczos(H.apply, guess, **self.opts)
        else:
            theta, u, nmv, rn, ok = davidson(H.apply, H.diagonal(), guess, **self.opts)
        ub = flat_to_blocks(H.layout, u)
        mid, Ab, Bb, trunc, kept = split_theta(ub, mps["bonds"][i], mps["bonds"][i + 2], D, direction, **self.dbss)
        mps["bonds"][i + 1] = mid
        mps["tensors"][i], mps["tensors"][i + 1] = Ab, Bb
        if direction == "fwd":
            mps["gauge"][i], mps["gauge"][i + 1] = "L", "C"
            self.L[i + 1] = grow(self.L[i], ham, mps["bonds"], Ab)
        else:
            mps["gauge"][i], mps["gauge"][i + 1] = "C", "R"
            self.R[i + 1] = grow(self.R[i + 2], ham, mps["bonds"], Bb)
        rec = dict(bond=i, dir=direction, energy=float(theta), n_matvec=nmv, residual=float(rn), converged=ok,
                   trunc_err=float(trunc), kept=int(kept), nsectors=len(mid), nnz=H.nnz)
        self.log.append(rec)
        return rec

    def sweep(self, D):
        recs = []
        for i in range(self.k - 1):
            recs.append(self._optimise(i, D, "fwd"))
        for i in range(self.k - 2, -1, -1):
            recs.append(self._optimise(i, D, "bwd"))
        return dict(energy_last=recs[-1]["energy"], energy_min=min(r["energy"] for r in recs), bonds=recs)

    def solve(self, D, eps_sweep, max_sweeps):
        """Sweeps until sweeps_converged (reading S34) or max_sweeps; returns the list of sweep results."""
        out = []
        while len(out) < max_sweeps:
            out.append(self.sweep(D))
            if sweeps_converged([r["energy_last"] for r in out], eps_sweep):
                break
        return out


# ----------------------------------------------------------------------------------------------------------------
# 1- and 2-RDM pass (C3 step 6; Eq. 9-10 under readings S2, S20)
# ----------------------------------------------------------------------------------------------------------------
def grow_normal(blk, ham, mps_bonds, tensor, two_index):
    """Blocking step that keeps only a+_P (and, if two_index, A_PQ and B_PS): what the RDM pass needs."""
    if blk.side == "L":
        p, nb = blk.b, blk.b + 1
    else:
        p, nb = blk.b - 1, blk.b - 1
    en = Enlarger(blk, ham, p)
    new = Block(blk.side, nb, blk.k, mps_bonds[nb])
    inside = new.inside()
    for a_, P in enumerate(inside):
        new.ops[("C", P)] = rotate(en.C(P), blk, tensor, new.basis)
        if two_index:
            for Q in inside[a_ + 1:]:
                new.ops[("A", P, Q)] = rotate(en.A(P, Q), blk, tensor, new.basis)
            for S in inside:
                new.ops[("B", P, S)] = rotate(en.B(P, S), blk, tensor, new.basis)
    return new


def _move_centre_right(mps, c):
    """QR of the centre tensor of site c per right sector: site c becomes left-orthonormal, R goes into site c+1."""
    bonds = mps["bonds"]
    ridx = {(n, s): j for j, (n, s, d) in enumerate(bonds[c + 1])}
    groups = {}
    for (li, a), t in mps["tensors"][c].items():
        n, s, _ = bonds[c][li]
        groups.setdefault(ridx[(n + SITE_Q[a][0], s + SITE_Q[a][1])], []).append((li, a))
    newA, Rf = {}, {}
    for mi, keys in groups.items():
        keys.sort()
        M = np.concatenate([mps["tensors"][c][key] for key in keys], axis=0)
        Q, R = np.linalg.qr(M)
        assert Q.shape[1] == M.shape[1], "rank-deficient centre: re-import a full-rank MPS"
        off = 0
        for key in keys:
            d = mps["tensors"][c][key].shape[0]
            newA[key] = np.ascontiguousarray(Q[off:off + d])
            off += d
        Rf[mi] = R
    mps["tensors"][c] = newA
    nxt = {}
    for (mi, b), t in mps["tensors"][c + 1].items():
        if mi in Rf:
            nxt[(mi, b)] = Rf[mi] @ t
    mps["tensors"][c + 1] = nxt


def _apply_right(Y, psi, bonds_l, bonds_r):
    """T[(l, s)] = psi[(l, s)] Y^T restricted to existing sectors, with the sign (-1)^{par_Y (N_l + N_s)};
    returns {(l, s): (r_out_idx, array[d_l, d_r_out])}."""
    ridx = {(n, s): j for j, (n, s, d) in enumerate(bonds_r)}
    out = {}
    for (li, a), t in psi.items():
        n, s, _ = bonds_l[li]
        ri = ridx[(n + SITE_Q[a][0], s + SITE_Q[a][1])]
        if Y is None:
            out[(li, a)] = (ri, t)
        elif ri in Y.blocks:
            ro, m = Y.blocks[ri]
            sgn = -1.0 if (Y.par and ((n + SITE_N[a]) & 1)) else 1.0
            out[(li, a)] = (ro, sgn * (t @ m.T))
    return out


def rdm12(h, eri, mps_in, want_2rdm=True):
    """gamma_pq = <E_pq>,  Gamma_pqrs = <sum_ss' a+_ps a+_rs' a_ss' a_qs>  of the normalised state of a
    right-canonical MPS whose norm sits in site 0.  Every spin-orbital element <a+_P a+_Q a_R a_S> (P<Q, S<R) is
    evaluated once, at the one-site centre c = the second smallest of its four site indices, as
    <psi_c| X_L (x) o_c (x) Y_R |psi_c> with X_L in {1, a+, a}, Y_R in {1, a+, a, A, A^T, B}."""
    ham = Ham(h, eri)
    k = ham.k
    n_so = 2 * k
    mps = dict(mps_in)
    mps["bonds"] = [list(b) for b in mps_in["bonds"]]
    mps["tensors"] = [dict(t) for t in mps_in["tensors"]]
    # right blocks R_k .. R_1 with normal operators
    Rb = {k: Block("R", k, k, mps["bonds"][k])}
    for b in range(k, 1, -1):
        Rb[b - 1] = grow_normal(Rb[b], ham, mps["bonds"], mps["tensors"][b - 1], want_2rdm)
    Lb = Block("L", 0, k, mps["bonds"][0])
    nrm2 = sum(np.sum(t * t) for t in mps["tensors"][0].values())
    g1 = np.zeros((n_so, n_so))
    g2 = np.zeros((n_so,) * 4) if want_2rdm else None
    site_of = lambda P: P >> 1

    site_mats = {}

    def site_mat(ops):
        key = tuple((P & 1, dag) for (P, dag) in ops)         # the 4x4 matrix depends only on spin and dagger
        if key not in site_mats:
            m = np.eye(4)
            for (P, dag) in ops:
                m = m @ (site_ann(P).T if dag else site_ann(P))
            site_mats[key] = m
        return site_mats[key]

    def right_op(RB, ops):
        if not ops:
            return None, 1.0
        if len(ops) == 1:
            (X, dag), = ops
            return (RB.ops[("C", X)] if dag else RB.ops[("C", X)].T()), 1.0
        (X, dx), (Y, dy) = ops
        if dx and dy:
            return (RB.ops[("A", X, Y)], 1.0) if X < Y else (RB.ops[("A", Y, X)], -1.0)
        if not dx and not dy:
            return (RB.ops[("A", Y, X)].T(), 1.0) if Y < X else (RB.ops[("A", X, Y)].T(), -1.0)
        assert dx and not dy
        return RB.ops[("B", X, Y)], 1.0

    for c in range(k):
        psi = mps["tensors"][c]
        bl, br = mps["bonds"][c], mps["bonds"][c + 1]
        RB = Rb[c + 1]
        # ---- gather the strings evaluated at this centre, grouped by their right-block factor ----------------
        groups = {}

        def add_string(ops, target):
            parts = [0 if site_of(P) < c else (1 if site_of(P) == c else 2) for (P, d) in ops]
            sign = 1.0
            order = list(range(len(ops)))
            for a_ in range(len(order)):                      # stable bubble sort by part, counting swaps
                for b_ in range(len(order) - 1 - a_):
                    if parts[order[b_]] > parts[order[b_ + 1]]:
                        order[b_], order[b_ + 1] = order[b_ + 1], order[b_]
                        sign = -sign
            lops = tuple(ops[j] for j in order if parts[j] == 0)
            cops = tuple(ops[j] for j in order if parts[j] == 1)
            rops = tuple(ops[j] for j in order if parts[j] == 2)
            groups.setdefault(rops, []).append((lops, cops, sign, target))

        for P in range(n_so):
            for S in range(n_so):
                if min(site_of(P), site_of(S)) == c:
                    add_string(((P, True), (S, False)), (P, S))
        if want_2rdm:
            # all (P<Q, S<R) whose second-smallest site is c, i.e. at most one operator left of c and at least two on
            # sites <= c.  Integer bookkeeping only: the pairs are binned by (#left of c, #on c) and only admissible bins
            # are combined (the same set as scanning every quadruple and testing sorted(sites)[1] == c; each string is
            # an independent assignment, so the visiting order does not matter).  Strings that change 2Sz are skipped:
            # their expectation value in an Sz eigenstate is zero (g2 starts at zero).
            bins = {}
            for P in range(n_so):
                for Q in range(P + 1, n_so):
                    nl = (site_of(P) < c) + (site_of(Q) < c)
                    nc = (site_of(P) == c) + (site_of(Q) == c)
                    if nl <= 1:
                        bins.setdefault((nl, nc), []).append((P, Q, spin_of(P) + spin_of(Q)))
            for (nl1, nc1), cre in bins.items():
                for (nl2, nc2), ann in bins.items():
                    if nl1 + nl2 > 1 or nl1 + nl2 + nc1 + nc2 < 2:
                        continue
                    for (P, Q, sc) in cre:
                        for (S, R, sa) in ann:
                            if sc == sa:
                                add_string(((P, True), (Q, True), (R, False), (S, False)), (P, Q, R, S))
        # ---- evaluate ------------------------------------------------------------------------------------------
        for rops, items in groups.items():
            Y, ycoef = right_op(RB, rops)
            T = _apply_right(Y, psi, bl, br)
            # N[(so, si)][(lo, li)] = sum_r psi[(lo,so)][:, r] T[(li,si)][:, r]^T  * (-1)^{par_o N_li}
            N = {}
            for (li, si), (ro, t) in T.items():
                for lo in range(len(bl)):
                    for so in range(4):
                        p2 = psi.get((lo, so))
                        if p2 is None:
                            continue
                        n, s, _ = bl[lo]
                        if (n + SITE_Q[so][0], s + SITE_Q[so][1]) != (br[ro][0], br[ro][1]):
                            continue
                        par_o = (SITE_N[so] - SITE_N[si]) & 1
                        sgn = -1.0 if (par_o and (bl[li][0] & 1)) else 1.0
                        N.setdefault((so, si), {})[(lo, li)] = sgn * (p2 @ t.T)
            cache = {}
            for (lops, cops, sign, target) in items:
                if lops not in cache:
                    val = np.zeros((4, 4))
                    if not lops:
                        for (so, si), blocks in N.items():
                            val[so, si] = sum(np.trace(m) for (lo, li), m in blocks.items() if lo == li)
                    else:
                        (PX, dag), = lops
                        X = Lb.ops[("C", PX)] if dag else Lb.ops[("C", PX)].T()
                        for (so, si), blocks in N.items():
                            acc = 0.0
                            for (lo, li), m in blocks.items():
                                if li in X.blocks and X.blocks[li][0] == lo:
                                    acc += np.sum(X.blocks[li][1] * m)
                            val[so, si] = acc
                    cache[lops] = val
                o = site_mat(cops)
                v = sign * ycoef * np.sum(o * cache[lops]) / nrm2
                if len(target) == 2:
                    g1[target] = v
                else:
                    P, Q, R, S = target
                    g2[P, Q, R, S] = v
                    g2[Q, P, R, S] = -v
                    g2[P, Q, S, R] = -v
                    g2[Q, P, S, R] = v
        if c < k - 1:
            _move_centre_right(mps, c)
            Lb = grow_normal(Lb, ham, mps["bonds"], mps["tensors"][c], False)
    gamma = g1[0::2, 0::2] + g1[1::2, 1::2]
    if not want_2rdm:
        return gamma, None
    # Gamma_pqrs = sum_{s,s'} G[(p s), (r s'), (s s'), (q s)]
    Gamma = np.zeros((k,) * 4)
    for s1 in (0, 1):
        for s2 in (0, 1):
            Gamma += g2[s1::2, s2::2, s2::2, s1::2].transpose(0, 3, 1, 2)
    return gamma, Gamma
