"""Seeded synthetic Hamiltonians: the five BASELINE.json configs plus small dense random cases for tests.

Inputs only - no DMRG arithmetic lives here.  Recipes:
  * PPP pi-Hamiltonian on a hexagonal carbon graph (C-C 1.40 A, t=-2.4 eV, U=11.26 eV, Ohno V_ij), in Hartree,
  * orbital rotation W = expm(kappa), kappa antisymmetric with N(0, 0.05) entries,
  * Fiedler ordering of |(pp|qq)|,
  * Fe-S-like dense Hamiltonian: (pq|rs) = sum_{K<80} L^K_pq L^K_rs.
The paper's own molecules (B3LYP/cc-pVDZ orbitals from ORCA) are not available; these
stand in for their shapes (half-filled PAH pi systems; a more-than-half-filled dense transition-metal-like CAS).
"""
import numpy as np

EV_PER_HARTREE = 27.211386245988
CC_BOND = 1.40          # Angstrom
PPP_T = -2.4            # eV
PPP_U = 11.26           # eV
OHNO_C = 14.397         # eV*Angstrom
CONFIG_SEED = 250320700  # + config number


def hex_graph(centres):
    """Sites/bonds of fused regular hexagons. centres: list of axial (q, r) hexagon coordinates.

    Hexagon centres sit on a triangular lattice of spacing sqrt(3)*1.40 A; vertices at angles 30+60j degrees;
    coincident vertices (1e-6 A) are merged; two sites are bonded iff their distance is 1.40 A.
    Returns (points [k,2], bonded [k,k] bool)."""
    a = CC_BOND
    s3 = np.sqrt(3.0)
    pts = []
    for (q, r) in centres:
        cx = s3 * a * (q + 0.5 * r)
        cy = 1.5 * a * r
        for j in range(6):
            ang = np.pi / 6 + j * np.pi / 3
            p = (cx + a * np.cos(ang), cy + a * np.sin(ang))
            if not any(abs(p[0] - u[0]) < 1e-6 and abs(p[1] - u[1]) < 1e-6 for u in pts):
                pts.append(p)
    pts = np.array(pts)
    dist = np.linalg.norm(pts[:, None, :] - pts[None, :, :], axis=2)
    bonded = np.abs(dist - a) < 1e-6
    return pts, bonded


def flake_centres(radius):
    """Hexagon flake: all axial (q, r) with max(|q|, |r|, |q+r|) <= radius (radius 1: coronene, 2: C54)."""
    out = []
    for q in range(-radius, radius + 1):
        for r in range(-radius, radius + 1):
            if max(abs(q), abs(r), abs(q + r)) <= radius:
                out.append((q, r))
    return out


def row_centres(n):
    """n linearly fused hexagons (n=2: naphthalene, n=20: the 82-site icosacene skeleton)."""
    return [(q, 0) for q in range(n)]


def ppp_integrals(pts, bonded):
    """PPP model H = sum_<ij>s t (a+_is a_js + h.c.) + U sum n_iu n_id + sum_{i<j} V_ij (n_i-1)(n_j-1) as
    (h, eri, e_core) in Hartree: h_ij = t (bonded), h_ii = -sum_{j!=i} V_ij, (ii|jj) = V_ij, (ii|ii) = U,
    e_core = sum_{i<j} V_ij.  Ohno: V_ij = U / sqrt(1 + (U r_ij / 14.397)^2), r in Angstrom, energies in eV."""
    k = len(pts)
    dist = np.linalg.norm(pts[:, None, :] - pts[None, :, :], axis=2)
    V = PPP_U / np.sqrt(1.0 + (PPP_U * dist / OHNO_C) ** 2)
    np.fill_diagonal(V, PPP_U)
    h = np.zeros((k, k))
    h[bonded] = PPP_T
    for i in range(k):
        h[i, i] = -(V[i].sum() - V[i, i])
    e_core = float(sum(V[i, j] for i in range(k) for j in range(i + 1, k)))
    eri = np.zeros((k, k, k, k))
    idx = np.arange(k)
    eri[idx[:, None], idx[:, None], idx[None, :], idx[None, :]] = V
    return h / EV_PER_HARTREE, eri / EV_PER_HARTREE, e_core / EV_PER_HARTREE


def _expm_antisym(kappa):
    """expm of a real antisymmetric matrix via the Hermitian eigen-decomposition of i*kappa."""
    w, v = np.linalg.eigh(1j * kappa)          # i*kappa is Hermitian; kappa = -i * v diag(w) v^H
    return np.real((v * np.exp(-1j * w)) @ v.conj().T)


def rotate_orbitals(h, eri, rng, std=0.05):
    """W = expm(kappa); kappa_pq ~ N(0, std) for p<q drawn row-major, kappa_qp = -kappa_pq.
    h' = W^T h W ; (pq|rs)' = sum W_ap W_bq W_cr W_ds (ab|cd).  Returns (h', eri', W)."""
    k = h.shape[0]
    kappa = np.zeros((k, k))
    iu = np.triu_indices(k, 1)
    kappa[iu] = rng.normal(0.0, std, size=len(iu[0]))
    kappa = kappa - kappa.T
    W = _expm_antisym(kappa)
    h2 = W.T @ h @ W
    e = np.tensordot(eri, W, axes=([3], [0]))                    # (a b c s)
    e = np.tensordot(e, W, axes=([2], [0]))                      # (a b s r)
    e = np.tensordot(e, W, axes=([1], [0]))                      # (a s r q)
    e = np.tensordot(e, W, axes=([0], [0]))                      # (s r q p)
    e2 = np.ascontiguousarray(e.transpose(3, 2, 1, 0))
    return h2, e2, W


def fiedler_order(eri):
    """Chain order = stable argsort of the Fiedler vector of the graph with weights |(pp|qq)| (p != q).
    Sign convention: the largest-magnitude entry of the vector is made positive."""
    k = eri.shape[0]
    idx = np.arange(k)
    w = np.abs(eri[idx[:, None], idx[:, None], idx[None, :], idx[None, :]]).copy()
    np.fill_diagonal(w, 0.0)
    lap = np.diag(w.sum(1)) - w
    _, vec = np.linalg.eigh(lap)
    f = vec[:, 1].copy()
    if f[np.argmax(np.abs(f))] < 0:
        f = -f
    return np.argsort(f, kind="stable")


def permute_orbitals(h, eri, perm):
    return (np.ascontiguousarray(h[np.ix_(perm, perm)]),
            np.ascontiguousarray(eri[np.ix_(perm, perm, perm, perm)]))


def fes_like(k, rng, n_chol=80):
    """Fe-S-like dense Hamiltonian (BASELINE.json configs[2]).  Draw order: for K in 0..n_chol-1 the entries
    L^K_pq (p<=q row-major) ~ N(0, 0.3*exp(-|p-q|/4)) mirrored; then h off-diagonals p<q ~ N(0, 0.1) row-major;
    then h diagonals ~ U[-2, 0].  Values are in Hartree."""
    iu = np.triu_indices(k)
    sd = 0.3 * np.exp(-np.abs(iu[0] - iu[1]) / 4.0)
    L = np.zeros((n_chol, k, k))
    for K in range(n_chol):
        vals = rng.normal(0.0, 1.0, size=len(iu[0])) * sd
        L[K][iu] = vals
        L[K] = L[K] + np.triu(L[K], 1).T
    eri = np.einsum("Kpq,Krs->pqrs", L, L, optimize=True)
    h = np.zeros((k, k))
    io = np.triu_indices(k, 1)
    h[io] = rng.normal(0.0, 0.1, size=len(io[0]))
    h = h + h.T
    h[np.arange(k), np.arange(k)] = rng.uniform(-2.0, 0.0, size=k)
    return h, np.ascontiguousarray(eri), 0.0


def random_dense(k, seed, n_chol=5, scale=0.4):
    """Small dense random real Hamiltonian with 8-fold symmetric (pq|rs) - test input only."""
    rng = np.random.default_rng(seed)
    L = rng.normal(size=(n_chol, k, k)) * scale
    L = L + L.transpose(0, 2, 1)
    eri = np.einsum("Kpq,Krs->pqrs", L, L, optimize=True)
    h = rng.normal(size=(k, k)) * scale
    h = h + h.T
    return h, np.ascontiguousarray(eri)


_CONFIGS = {
    1: dict(name="naphthalene CAS(10,10) PPP", centres=lambda: row_centres(2), D=64, sweeps=4),
    2: dict(name="coronene CAS(24,24) PPP", centres=lambda: flake_centres(1), D=512, sweeps=6),
    3: dict(name="Fe-S-like CAS(30,20) dense Cholesky", centres=None, D=1024, sweeps=8),
    4: dict(name="circumcoronene CAS(54,54) PPP", centres=lambda: flake_centres(2), D=4096, sweeps=1),
    5: dict(name="icosacene-skeleton CAS(82,82) PPP", centres=lambda: row_centres(20), D=2048, sweeps=1),
    # not a BASELINE config: the open-shell second workload of SURVEY.md 8(f) rank 4 (Fe-S clusters with
    # S = 5/2) - the Fe-S-like dense Hamiltonian of config 3 (same recipe, its own seed) with an odd electron count in
    # the 2Sz = 5 member of a sextet
    6: dict(name="Fe-S-like open-shell CAS(29,20) dense Cholesky, 2Sz=5", centres=None, D=512, sweeps=4),
}


def make_config(c, rotate=True):
    """BASELINE.json configs[c-1] as concrete arrays.
    Returns dict(name, k, n_elec, two_sz, h, eri, e_core, D, sweeps, seed, order)."""
    spec = _CONFIGS[c]
    seed = CONFIG_SEED + c
    rng = np.random.default_rng(seed)
    two_sz = 0
    if c in (3, 6):
        k, n_elec = 20, (30 if c == 3 else 29)
        two_sz = 0 if c == 3 else 5
        h, eri, e_core = fes_like(k, rng)
        order = np.arange(k)
    else:
        pts, bonded = hex_graph(spec["centres"]())
        k = len(pts)
        n_elec = k
        h, eri, e_core = ppp_integrals(pts, bonded)
        if rotate:
            h, eri, _ = rotate_orbitals(h, eri, rng)
        order = fiedler_order(eri)
        h, eri = permute_orbitals(h, eri, order)
    return dict(name=spec["name"], k=k, n_elec=n_elec, two_sz=two_sz, h=h, eri=eri, e_core=e_core,
                D=spec["D"], sweeps=spec["sweeps"], seed=seed, order=order)
