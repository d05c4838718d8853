"""Pins for oracle tier 1 (brute-force FCI): closed forms, dense Jordan-Wigner matrices, invariants.
Citations: DESIGN.md C5 table; PAPER.md:52-68 (Hamiltonian), 91-93 (RDMs), 107 (site basis), 122-125 (MPS)."""
import itertools
import math

import numpy as np
import pytest

from oracle import fci
from synth import (hex_graph, row_centres, ppp_integrals, rotate_orbitals, fiedler_order, permute_orbitals,
                   random_dense, random_mps, make_config)
from synth.hamiltonians import EV_PER_HARTREE, PPP_T, PPP_U, OHNO_C, CC_BOND


def _ppp_chain(n):
    pts = np.array([[CC_BOND * i, 0.0] for i in range(n)])
    d = np.abs(pts[:, None, 0] - pts[None, :, 0])
    return pts, np.abs(d - CC_BOND) < 1e-9


def test_ppp_dimer_closed_form():
    # two sites, two electrons, singlet: E_el + E_core = (U-V)/2 - sqrt(((U-V)/2)^2 + 4 t^2)
    pts, bonded = _ppp_chain(2)
    h, eri, ecore = ppp_integrals(pts, bonded)
    V = PPP_U / math.sqrt(1 + (PPP_U * CC_BOND / OHNO_C) ** 2)
    assert abs(V - 7.59336) < 1e-5                     # Ohno V at 1.40 A, eV (DESIGN.md generator pin)
    exact = ((PPP_U - V) / 2 - math.sqrt(((PPP_U - V) / 2) ** 2 + 4 * PPP_T ** 2)) / EV_PER_HARTREE
    sp = fci.FCISpace(2, 2, 0)
    e, _ = sp.ground_state(h, eri)
    assert abs(e + ecore - exact) < 1e-12


@pytest.mark.parametrize("centres,k,expect", [(row_centres(1), 6, 8.0), (row_centres(2), 10, 13.6832)])
def test_hueckel_limit(centres, k, expect):
    # U = V = 0: E = 2 * sum of occupied Hueckel levels = -expect*|t| (benzene 8|t|, naphthalene 13.6832|t|)
    pts, bonded = hex_graph(centres)
    assert len(pts) == k
    h = np.zeros((k, k))
    h[bonded] = PPP_T / EV_PER_HARTREE
    eri = np.zeros((k,) * 4)
    w = np.linalg.eigvalsh(h)
    e_det = 2 * w[:k // 2].sum()
    assert abs(e_det * EV_PER_HARTREE + expect * abs(PPP_T)) < 2e-4 * abs(PPP_T)
    if k <= 6:
        sp = fci.FCISpace(k, k, 0)
        e, _ = sp.ground_state(h, eri)
        assert abs(e - e_det) < 1e-11
        # any orbital rotation leaves it unchanged
        h2, eri2, _ = rotate_orbitals(h, eri, np.random.default_rng(3))
        e2, _ = sp.ground_state(h2, eri2)
        assert abs(e2 - e_det) < 1e-11


def test_sector_dimension_config1():
    assert len(fci.sector_dets(10, 10, 0)) == math.comb(10, 5) ** 2 == 63504


@pytest.mark.parametrize("k,n,s2", [(3, 3, 1), (3, 4, 0), (4, 4, 0), (4, 5, -1), (4, 6, 2)])
def test_sector_fci_vs_dense_jordan_wigner(k, n, s2):
    h, eri = random_dense(k, 100 + k + n)
    H = fci.dense_jw_hamiltonian(h, eri)
    sp = fci.FCISpace(k, n, s2)
    Hs = sp.dense_h(h, eri)
    idx = sp.dets.astype(np.int64)
    assert np.abs(Hs - H[np.ix_(idx, idx)]).max() < 1e-12
    # the full-space H does not connect the sector to anything else
    mask = np.ones(H.shape[0], bool)
    mask[idx] = False
    assert np.abs(H[np.ix_(mask, idx)]).max() < 1e-12


def test_spin_orbital_form_equals_spatial_form():
    k = 3
    h, eri = random_dense(k, 5)
    a = fci.jw_annihilators(2 * k)
    ad = [x.T for x in a]
    t, v = fci.spin_orbital_integrals(h, eri)
    H = sum(t[P, Q] * ad[P] @ a[Q] for P in range(2 * k) for Q in range(2 * k))
    for P, Q, R, S in itertools.product(range(2 * k), repeat=4):
        if v[P, Q, R, S] != 0:
            H = H + 0.5 * v[P, Q, R, S] * ad[P] @ ad[Q] @ a[R] @ a[S]
    assert np.abs(H - fci.dense_jw_hamiltonian(h, eri)).max() < 1e-12


def test_rotation_and_ordering_invariance_of_fci_energy():
    pts, bonded = hex_graph(row_centres(1))
    h, eri, _ = ppp_integrals(pts, bonded)
    sp = fci.FCISpace(6, 6, 0)
    e0, _ = sp.ground_state(h, eri)
    h2, eri2, W = rotate_orbitals(h, eri, np.random.default_rng(11))
    assert np.abs(W.T @ W - np.eye(6)).max() < 1e-14
    order = fiedler_order(eri2)
    h3, eri3 = permute_orbitals(h2, eri2, order)
    e3, _ = sp.ground_state(h3, eri3)
    assert abs(e3 - e0) < 1e-10
    # 8-fold symmetry of the rotated integrals
    for perm in [(1, 0, 2, 3), (0, 1, 3, 2), (2, 3, 0, 1)]:
        assert np.abs(eri3 - eri3.transpose(perm)).max() < 1e-13


def test_rdm_invariants_and_energy_formula():
    k, n, s2 = 4, 5, 1
    h, eri = random_dense(k, 21)
    sp = fci.FCISpace(k, n, s2)
    e, c = sp.ground_state(h, eri)
    g, G = sp.rdm12(c)
    assert abs(np.trace(g) - n) < 1e-12
    assert np.abs(np.einsum("pqrr->pq", G) - (n - 1) * g).max() < 1e-12
    assert abs(np.einsum("pprr->", G) - n * (n - 1)) < 1e-11
    assert np.abs(G - G.transpose(2, 3, 0, 1)).max() < 1e-12
    assert np.abs(G - G.transpose(1, 0, 3, 2)).max() < 1e-12
    w = np.linalg.eigvalsh(g)
    assert w.min() > -1e-12 and w.max() < 2 + 1e-12
    assert abs(np.einsum("pq,pq", h, g) + 0.5 * np.einsum("pqrs,pqrs", eri, G) - e) < 1e-11
    # literal definition of Gamma through dense Jordan-Wigner matrices, spin-orbital string form
    a = fci.jw_annihilators(2 * k)
    ad = [x.T for x in a]
    psi = np.zeros(1 << (2 * k))
    psi[sp.dets.astype(np.int64)] = c
    for (p, q, r, s) in [(0, 1, 2, 3), (1, 1, 2, 0), (3, 0, 0, 2), (2, 2, 2, 2)]:
        val = sum(psi @ ad[2 * p + x] @ ad[2 * r + y] @ a[2 * s + y] @ a[2 * q + x] @ psi
                  for x in (0, 1) for y in (0, 1))
        assert abs(val - G[p, q, r, s]) < 1e-12


def test_closed_shell_rdm_closed_form():
    # U = V = 0 single determinant: gamma^2 = 2 gamma,  Gamma_pqrs = gamma_pq gamma_rs - 1/2 gamma_ps gamma_rq
    pts, bonded = hex_graph(row_centres(1))
    k = 6
    h = np.zeros((k, k))
    h[bonded] = -1.0
    h2, eri2, _ = rotate_orbitals(h, np.zeros((k,) * 4), np.random.default_rng(2))
    sp = fci.FCISpace(k, 6, 0)
    e, c = sp.ground_state(h2, eri2)
    g, G = sp.rdm12(c)
    assert np.abs(g @ g - 2 * g).max() < 1e-10
    ref = np.einsum("pq,rs->pqrs", g, g) - 0.5 * np.einsum("ps,rq->pqrs", g, g)
    assert np.abs(G - ref).max() < 1e-10


def test_mps_expansion_norm_and_heff_symmetry():
    k, n, s2 = 6, 6, 0
    h, eri = random_dense(k, 9)
    sp = fci.FCISpace(k, n, s2)
    mps = random_mps(k, n, s2, 12, seed=4, gauge="R")
    c = fci.mps_to_ci(mps, sp)
    assert abs(np.linalg.norm(c) - 1.0) < 1e-12          # right-canonical MPS with 1x1 left boundary
    i = 2
    mps2 = random_mps(k, n, s2, 12, seed=5, gauge="LR:%d" % i)
    layout, nnz = fci.heff_layout(mps2, i)
    rng = np.random.default_rng(0)
    x, z = rng.normal(size=nnz), rng.normal(size=nnz)
    hx = fci.heff_apply_bruteforce(mps2, i, h, eri, x, sp)
    hz = fci.heff_apply_bruteforce(mps2, i, h, eri, z, sp)
    assert abs(z @ hx - x @ hz) < 1e-11 * (np.linalg.norm(hx) * np.linalg.norm(z))
    # P is an isometry: ||P x|| = ||x||  -> Rayleigh quotient bounded by the FCI spectrum
    e0, _ = sp.ground_state(h, eri)
    assert x @ hx / (x @ x) >= e0 - 1e-10


@pytest.mark.slow
def test_config1_fci_energy_survey_crosscheck():
    # E_el + E_core = -0.8822829988 Eh, E_core = 8.5092529943 Eh; seed independent.
    cfg = make_config(1)
    assert abs(cfg["e_core"] - 8.5092529943) < 1e-9
    sp = fci.FCISpace(10, 10, 0)
    e, _ = sp.ground_state(cfg["h"], cfg["eri"], tol=1e-11)
    assert abs(e + cfg["e_core"] - (-0.8822829988)) < 2e-9
