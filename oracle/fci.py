"""ORACLE, tier 1 (test infrastructure - never imported by the product path): brute-force full CI.

Plain definitions, FP64, numpy/scipy.sparse only.  What is defined here, and from where:

  * H_el = sum_pq h_pq E_pq + 1/2 sum_pqrs (pq|rs) (E_pq E_rs - delta_qr E_ps),  E_pq = sum_s a+_ps a_qs
    PAPER.md:52-68 (Eq. 1-5) under reading S1 of DESIGN.md (the printed Eq. 1-3 lack the 1/2 and pair the indices
    inconsistently with Eq. 5; the Coulomb Hamiltonian with chemists' (pq|rs) of Eq. 5 is taken).
  * gamma_pq = <E_pq> (Eq. 9);  Gamma_pqrs = <E_pq E_rs - delta_qr E_ps> (Eq. 10 under
    reading S2: index order chosen so that E = sum h gamma + 1/2 sum (pq|rs) Gamma).
  * site basis |0>, |dn>, |up>, |up dn>; determinant |n> = prod_{P ascending} (a+_P)^{n_P} |0>
    with spin-orbital index P = 2p + [spin = dn] (readings S3, S4), stored as bit P of an integer.
  * MPS -> CI expansion: psi_{i_1..i_k} = A^{i_1} ... A^{i_k} (Eq. 14).
  * H_eff x := P^T H_el P x at a two-site bond (plain definition, C2).

Pins (tests/test_oracle_fci.py): PPP dimer closed form, Hueckel limits, dense Jordan-Wigner matrices for k<=4,
rotation invariance, sector dimension C(10,5)^2, RDM invariants, closed-shell Gamma formula.
"""
import itertools
import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as sla

SITE_Q = ((0, 0), (1, -1), (1, 1), (2, 0))            # (N, 2Sz) of the four site states
SITE_BITS = (0b00, 0b10, 0b01, 0b11)                  # bit0 = up (P=2p), bit1 = down (P=2p+1)


def popcount(x):
    x = np.asarray(x, dtype=np.uint64)
    c = np.zeros(x.shape, dtype=np.int64)
    y = x.copy()
    while np.any(y):
        c += (y & np.uint64(1)).astype(np.int64)
        y >>= np.uint64(1)
    return c


def sector_dets(k, n_elec, two_sz):
    """All determinants (bitmasks over 2k spin orbitals) with N = n_elec and 2Sz = two_sz, ascending."""
    n_up = (n_elec + two_sz) // 2
    n_dn = (n_elec - two_sz) // 2
    assert n_up + n_dn == n_elec and 0 <= n_up <= k and 0 <= n_dn <= k
    ups = [sum(1 << (2 * o) for o in c) for c in itertools.combinations(range(k), n_up)]
    dns = [sum(1 << (2 * o + 1) for o in c) for c in itertools.combinations(range(k), n_dn)]
    dets = np.array(sorted(u | d for u in ups for d in dns), dtype=np.uint64)
    return dets


class FCISpace:
    """Determinant basis of one (N, 2Sz) sector and the spin-summed excitation operators E_pq on it."""

    def __init__(self, k, n_elec, two_sz):
        self.k, self.n_elec, self.two_sz = k, n_elec, two_sz
        self.dets = sector_dets(k, n_elec, two_sz)
        self.dim = len(self.dets)
        self._E = {}

    def index_of(self, dets):
        idx = np.searchsorted(self.dets, dets)
        idx = np.clip(idx, 0, self.dim - 1)
        ok = self.dets[idx] == dets
        return idx, ok

    def _so_excitation(self, P, Q):
        """a+_P a_Q on the sector basis as (rows, cols, signs)."""
        d = self.dets
        one = np.uint64(1)
        occQ = ((d >> np.uint64(Q)) & one) == 1
        cols = np.nonzero(occQ)[0]
        s1 = d[cols] ^ (one << np.uint64(Q))
        sg = 1 - 2 * (popcount(s1 & ((one << np.uint64(Q)) - one)) & 1)
        freeP = ((s1 >> np.uint64(P)) & one) == 0
        cols, s1, sg = cols[freeP], s1[freeP], sg[freeP]
        sg = sg * (1 - 2 * (popcount(s1 & ((one << np.uint64(P)) - one)) & 1))
        s2 = s1 | (one << np.uint64(P))
        rows, ok = self.index_of(s2)
        assert np.all(ok)
        return rows, cols, sg.astype(np.float64)

    def E(self, p, q):
        """E_pq = a+_{p up} a_{q up} + a+_{p dn} a_{q dn} as a sparse matrix on the sector."""
        key = (p, q)
        if key not in self._E:
            r1, c1, v1 = self._so_excitation(2 * p, 2 * q)
            r2, c2, v2 = self._so_excitation(2 * p + 1, 2 * q + 1)
            self._E[key] = sp.csr_matrix((np.concatenate([v1, v2]),
                                          (np.concatenate([r1, r2]), np.concatenate([c1, c2]))),
                                         shape=(self.dim, self.dim))
        return self._E[key]

    def apply_h(self, h, eri, c):
        """sigma = H_el c by the definition  sum h E_pq + 1/2 sum (pq|rs)(E_pq E_rs - delta_qr E_ps)."""
        k = self.k
        D = np.empty((k, k, self.dim))
        for r in range(k):
            for s in range(k):
                D[r, s] = self.E(r, s) @ c
        heff = h - 0.5 * np.einsum("prrs->ps", eri)            # the -delta_qr E_ps part
        G = 0.5 * np.tensordot(eri, D, axes=([2, 3], [0, 1]))   # G_pq = 1/2 sum_rs (pq|rs) E_rs c
        out = np.tensordot(heff, D, axes=([0, 1], [0, 1]))
        for p in range(k):
            for q in range(k):
                out += self.E(p, q) @ G[p, q]
        return out

    def linear_operator(self, h, eri):
        return sla.LinearOperator((self.dim, self.dim), matvec=lambda c: self.apply_h(h, eri, c), dtype=np.float64)

    def dense_h(self, h, eri):
        """Explicit sector Hamiltonian (small sectors only)."""
        eye = np.eye(self.dim)
        return np.stack([self.apply_h(h, eri, eye[:, j]) for j in range(self.dim)], axis=1)

    def ground_state(self, h, eri, tol=1e-12, seed=0):
        """Lowest eigenpair of H_el in the sector (Eq. 15, without the MPS restriction)."""
        if self.dim <= 600:
            w, v = np.linalg.eigh(self.dense_h(h, eri))
            return float(w[0]), v[:, 0]
        rng = np.random.default_rng(seed)
        w, v = sla.eigsh(self.linear_operator(h, eri), k=1, which="SA", tol=tol, v0=rng.normal(size=self.dim),
                         ncv=40, maxiter=5000)
        return float(w[0]), v[:, 0]

    def rdm12(self, c):
        """gamma_pq = <E_pq>, Gamma_pqrs = <E_pq E_rs> - delta_qr <E_ps> for the normalised vector c."""
        k = self.k
        c = c / np.linalg.norm(c)
        D = np.empty((k, k, self.dim))
        for r in range(k):
            for s in range(k):
                D[r, s] = self.E(r, s) @ c
        gamma = np.tensordot(D, c, axes=([2], [0]))
        Dm = D.reshape(k * k, self.dim)
        # <E_pq E_rs> = (E_qp c) . (E_rs c)   because E_pq^T = E_qp
        EE = (Dm @ Dm.T).reshape(k, k, k, k).transpose(1, 0, 2, 3)
        Gamma = EE.copy()
        for q in range(k):
            Gamma[:, q, q, :] -= gamma
        return gamma, Gamma


# ----------------------------------------------------------------------------------------------------------------
# dense Jordan-Wigner matrices on the whole Fock space (k <= 5): the most literal form of the definitions
# ----------------------------------------------------------------------------------------------------------------
def jw_annihilators(n_so):
    """a_P for P = 0..n_so-1 as dense 2^n x 2^n matrices; basis index = occupation bitmask with bit P = n_P and
    |n> = prod_{P ascending} (a+_P)^{n_P}|0>, hence a_P|n> = (-1)^{sum_{P'<P} n_P'} |n - e_P>."""
    dim = 1 << n_so
    ops = []
    for P in range(n_so):
        m = np.zeros((dim, dim))
        for n in range(dim):
            if (n >> P) & 1:
                sign = (-1) ** bin(n & ((1 << P) - 1)).count("1")
                m[n ^ (1 << P), n] = sign
        ops.append(m)
    return ops


def spin_orbital_integrals(h, eri):
    """t_PQ = h_pq delta_ss',  v_PQRS = (ps|qr) delta(sP,sS) delta(sQ,sR) so that
    H_el = sum t_PQ a+_P a_Q + 1/2 sum v_PQRS a+_P a+_Q a_R a_S  (C1)."""
    k = h.shape[0]
    n = 2 * k
    t = np.zeros((n, n))
    v = np.zeros((n, n, n, n))
    for s in (0, 1):
        t[s::2, s::2] = h
    for s1 in (0, 1):
        for s2 in (0, 1):
            # P,S carry spin s1 ; Q,R carry spin s2 ; v[P,Q,R,S] = eri[p,s,q,r]
            v[s1::2, s2::2, s2::2, s1::2] = eri.transpose(0, 2, 3, 1)
    return t, v


def dense_jw_hamiltonian(h, eri):
    """H_el on the full Fock space from the spatial-orbital definition (E_pq form)."""
    k = h.shape[0]
    a = jw_annihilators(2 * k)
    ad = [x.T for x in a]
    E = [[ad[2 * p] @ a[2 * q] + ad[2 * p + 1] @ a[2 * q + 1] for q in range(k)] for p in range(k)]
    H = np.zeros_like(a[0])
    for p in range(k):
        for q in range(k):
            H += h[p, q] * E[p][q]
    for p, q, r, s in itertools.product(range(k), repeat=4):
        H += 0.5 * eri[p, q, r, s] * (E[p][q] @ E[r][s] - (q == r) * E[p][s])
    return H


# ----------------------------------------------------------------------------------------------------------------
# MPS <-> CI and the plain definition of H_eff x
# ----------------------------------------------------------------------------------------------------------------
def _grow_left(mps, upto):
    """States of the block of sites [0, upto): {sector idx on bond `upto`: (bitmasks [n], amps [n, dim])} with
    amps[det, alpha] = (A^{s_0} ... A^{s_{upto-1}})[0, alpha]  (Eq. 14)."""
    cur = {0: (np.zeros(1, dtype=np.uint64), np.ones((1, 1)))}
    for p in range(upto):
        index = {(n, s): i for i, (n, s, d) in enumerate(mps["bonds"][p + 1])}
        acc = {}
        for li, (bits, amps) in cur.items():
            n, s, _ = mps["bonds"][p][li]
            for st in range(4):
                blk = mps["tensors"][p].get((li, st))
                if blk is None:
                    continue
                ri = index[(n + SITE_Q[st][0], s + SITE_Q[st][1])]
                nb = bits | (np.uint64(SITE_BITS[st]) << np.uint64(2 * p))
                acc.setdefault(ri, []).append((nb, amps @ blk))
        cur = {ri: (np.concatenate([x[0] for x in lst]), np.concatenate([x[1] for x in lst], axis=0))
               for ri, lst in acc.items()}
    return cur


def _grow_right(mps, frm):
    """States of the block of sites [frm, k): {sector idx on bond `frm`: (bitmasks [n], amps [dim, n])} with
    amps[alpha, det] = (B^{s_frm} ... B^{s_{k-1}})[alpha, 0]."""
    k = mps["k"]
    cur = {0: (np.zeros(1, dtype=np.uint64), np.ones((1, 1)))}
    for p in range(k - 1, frm - 1, -1):
        index = {(n, s): i for i, (n, s, d) in enumerate(mps["bonds"][p + 1])}
        acc = {}
        for li, (n, s, _) in enumerate(mps["bonds"][p]):
            for st in range(4):
                blk = mps["tensors"][p].get((li, st))
                if blk is None:
                    continue
                ri = index[(n + SITE_Q[st][0], s + SITE_Q[st][1])]
                if ri not in cur:
                    continue
                bits, amps = cur[ri]
                nb = bits | (np.uint64(SITE_BITS[st]) << np.uint64(2 * p))
                acc.setdefault(li, []).append((nb, blk @ amps))
        cur = {li: (np.concatenate([x[0] for x in lst]), np.concatenate([x[1] for x in lst], axis=1))
               for li, lst in acc.items()}
    return cur


def mps_to_ci(mps, space):
    """CI vector of the state the MPS represents (not normalised): Eq. 14 written out."""
    left = _grow_left(mps, mps["k"])
    c = np.zeros(space.dim)
    for ri, (bits, amps) in left.items():
        idx, ok = space.index_of(bits)
        assert np.all(ok)
        np.add.at(c, idx, amps[:, 0])
    return c


def heff_layout(mps, i):
    """psi blocks at two-site bond i: list of (l_idx, s_i, s_j, r_idx, rows, cols, offset), ordered by
    (l_idx, s_i, s_j); left sectors from bond i, right sectors from bond i+2."""
    bl, br = mps["bonds"][i], mps["bonds"][i + 2]
    rindex = {(n, s): j for j, (n, s, d) in enumerate(br)}
    out, off = [], 0
    for li, (n, s, dl) in enumerate(bl):
        for si in range(4):
            for sj in range(4):
                key = (n + SITE_Q[si][0] + SITE_Q[sj][0], s + SITE_Q[si][1] + SITE_Q[sj][1])
                if key in rindex:
                    ri = rindex[key]
                    dr = br[ri][2]
                    out.append((li, si, sj, ri, dl, dr, off))
                    off += dl * dr
    return out, off


def heff_apply_bruteforce(mps, i, h, eri, x, space):
    """y = P^T H_el P x: expand x with the block states of sites < i and > i+1 to a CI vector, apply the FCI
    Hamiltonian, contract back with the same block states (C2)."""
    layout, nnz = heff_layout(mps, i)
    assert x.shape == (nnz,)
    left = _grow_left(mps, i)
    right = _grow_right(mps, i + 2)
    c = np.zeros(space.dim)
    maps = []
    for (li, si, sj, ri, dl, dr, off) in layout:
        if li not in left or ri not in right:
            maps.append(None)
            continue
        lb, la = left[li]
        rb, ra = right[ri]
        mid = (np.uint64(SITE_BITS[si]) << np.uint64(2 * i)) | (np.uint64(SITE_BITS[sj]) << np.uint64(2 * i + 2))
        dets = (lb[:, None] | rb[None, :] | mid).ravel()
        idx, ok = space.index_of(dets)
        assert np.all(ok)
        maps.append((idx, la, ra))
        blk = x[off:off + dl * dr].reshape(dl, dr)
        np.add.at(c, idx, (la @ blk @ ra).ravel())
    sigma = space.apply_h(h, eri, c)
    y = np.zeros(nnz)
    for (li, si, sj, ri, dl, dr, off), m in zip(layout, maps):
        if m is None:
            continue
        idx, la, ra = m
        S = sigma[idx].reshape(la.shape[0], ra.shape[1])
        y[off:off + dl * dr] = (la.T @ S @ ra.T).ravel()
    return y
