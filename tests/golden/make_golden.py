"""Writes the stored expected values under tests/golden/ by calling ONLY oracle/ on the seeded generators of synth/.
Nothing here imports the CUDA package.  Each file records the command that wrote it and how long the oracle took.

  python tests/golden/make_golden.py fci
      config1_fci.txt - BASELINE.json configs[0] (PPP naphthalene CAS(10,10), 2Sz = 0, FCI dimension 63504, readings
      S6-S9 of DESIGN.md): E_core, E_el(FCI), E_total, Tr gamma and the natural occupations of the FCI 1-RDM
      (Eq. 9) from oracle/fci.py.  The total energy is seed independent (invariant under the exp(kappa)
      rotation) and agrees with the survey's independent probe value -0.8822829988 Eh.

  python tests/golden/make_golden.py heff CFG D BOND [BOND ...]
      heff_cfgC_DD.npz - y = H_eff x (y = P^T H P x, Eq. 1-5 and 122-130 Eq. 14-15; C2),
      diag(H_eff) and the oracle's own GEMM-flop count at the listed two-site bonds of BASELINE config CFG at bond
      dimension D, from oracle/dmrg.py (tier 2) on its own environments.  Inputs: the "dual gauge" pair of seeded MPS
      (left-orthonormal A with seed s, right-orthonormal B with seed s + 1 on one sector plan, s = config seed + 2000)
      and x = normalised N(0,1) vector from default_rng(1000 + bond) - tests/test_gpu_golden.py rebuilds the same
      inputs for the CUDA library.  The plain Python oracle cannot reach the configs' own D (4096 / 2048) on k = 54 /
      82 in bounded time; the files say which D it did reach and how long that took.

  python tests/golden/make_golden.py sweep CFG D NSWEEPS [DINIT [NBONDS]]
      sweep_cfgC_DD.json - per-bond Davidson energies, kept bond dimension, sector count and truncation error of
      NSWEEPS two-site sweeps (readings S12-S18, Davidson tolerance 1e-10 as in S13) from oracle.dmrg.SweepEngine on
      random_mps(seed = config seed + 1000, gauge R, D = DINIT or D).  With NBONDS (k = 54): only the first NBONDS bond
      steps of the first forward pass.

  python tests/golden/make_golden.py rdm CFG D [NSAMPLE]
      rdm_cfgC_DD.npz - gamma and Gamma (Eq. 9-10, readings S2 / S20) of random_mps(seed = 900 + CFG,
      gauge R) from oracle.dmrg.rdm12; with NSAMPLE (k = 54: Gamma has 8.5e6 entries) a seeded sample of Gamma plus
      the full-array scalars sum Gamma^2 and sum_pr Gamma_pprr instead of the whole array.

CFG 1-5 are BASELINE.json's configs; CFG 6 is the open-shell second workload of synth/ (Fe-S-like CAS(29,20), 2Sz = 5;
SURVEY.md 8(f) rank 4).
"""
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from oracle import dmrg as odmrg  # noqa: E402
from oracle import fci  # noqa: E402
from synth import dual_gauge_mps, make_config, random_mps  # noqa: E402


def golden_fci():
    cfg = make_config(1)
    sp = fci.FCISpace(cfg["k"], cfg["n_elec"], 0)
    e, c = sp.ground_state(cfg["h"], cfg["eri"], tol=1e-12)
    g, G = sp.rdm12(c)
    occ = np.sort(np.linalg.eigvalsh(g))[::-1]
    with open(os.path.join(HERE, "config1_fci.txt"), "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/fci.py (brute-force FCI, dim %d)\n" % sp.dim)
        f.write("e_core %.10f\n" % cfg["e_core"])
        f.write("e_el_fci %.10f\n" % e)
        f.write("e_total_fci %.10f\n" % (e + cfg["e_core"]))
        f.write("trace_gamma %.10f\n" % np.trace(g))
        f.write("natural_occupations " + " ".join("%.8f" % x for x in occ) + "\n")


def golden_heff(cid, D, bonds):
    cfg = make_config(cid)
    A, B = dual_gauge_mps(cfg["k"], cfg["n_elec"], cfg["two_sz"], D, cfg["seed"] + 2000)
    ham = odmrg.Ham(cfg["h"], cfg["eri"])
    t0 = time.time()
    oL = odmrg.build_left(A, ham, max(bonds))
    oR = odmrg.build_right(B, ham, min(bonds) + 2)
    t_env = time.time() - t0
    out = dict(bonds=np.array(bonds), D=D, config=cid, mps_seed=cfg["seed"] + 2000)
    secs = {}
    for i in bonds:
        t0 = time.time()
        H = odmrg.Heff(oL[i], oR[i + 2], ham, i)
        x = np.random.default_rng(1000 + i).normal(size=H.nnz)
        x /= np.linalg.norm(x)
        out["y_%d" % i] = H.apply(x)
        out["diag_%d" % i] = H.diagonal()
        out["nnz_%d" % i] = H.nnz
        out["nterms_%d" % i] = len(H.terms)
        out["gemm_flops_%d" % i] = H.gemm_flops()
        out["layout_%d" % i] = np.array([b[:6] for b in H.layout], dtype=np.int64)
        secs[i] = time.time() - t0
        print("config %d D=%d bond %d: nnz=%d, %.0f s" % (cid, D, i, H.nnz, secs[i]), flush=True)
    out["note"] = ("written by `python tests/golden/make_golden.py heff %d %d %s` from oracle/dmrg.py; oracle time: "
                   "environments %.0f s, per bond %s s on %d host cores" %
                   (cid, D, " ".join(map(str, bonds)), t_env, {i: round(s) for i, s in secs.items()}, os.cpu_count()))
    np.savez_compressed(os.path.join(HERE, "heff_cfg%d_D%d.npz" % (cid, D)), **out)
    print(out["note"], flush=True)


def golden_sweep(cid, D, nsweeps, Dinit, nbonds=0):
    """nbonds > 0 (large k, where a whole oracle sweep takes many hours): only the first nbonds bond steps of the forward
    pass of the first sweep, in the sweep's own order (SweepEngine._optimise, the step sweep() itself calls); they do not
    depend on the later ones."""
    cfg = make_config(cid)
    k, n = cfg["k"], cfg["n_elec"]
    mps = random_mps(k, n, cfg["two_sz"], Dinit, seed=cfg["seed"] + 1000, gauge="R")
    t0 = time.time()
    eng = odmrg.SweepEngine(cfg["h"], cfg["eri"], mps, davidson_tol=1e-10)
    print("right environments built, %.0f s" % (time.time() - t0), flush=True)
    sweeps = []
    if nbonds:
        recs = []
        for i in range(nbonds):
            recs.append(eng._optimise(i, D, "fwd"))
            print("config %d D=%d bond %d: E = %.12f, %d matvecs (%.0f s)" % (cid, D, i, recs[-1]["energy"], recs[-1]["n_matvec"], time.time() - t0), flush=True)
        sweeps.append(dict(energy_last=None, energy_min=None, bonds=recs))
    for s in range(0 if nbonds else nsweeps):
        r = eng.sweep(D)
        sweeps.append(r)
        print("config %d D=%d sweep %d: E_last = %.12f (%.0f s)" % (cid, D, s, r["energy_last"], time.time() - t0), flush=True)
    note = ("written by `python tests/golden/make_golden.py sweep %d %d %d %d%s` from oracle.dmrg.SweepEngine "
            "(Davidson tol 1e-10); oracle time %.0f s on %d host cores" % (cid, D, nsweeps, Dinit, " %d" % nbonds if nbonds else "", time.time() - t0, os.cpu_count()))
    with open(os.path.join(HERE, "sweep_cfg%d_D%d.json" % (cid, D)), "w") as f:
        json.dump(dict(note=note, config=cid, D=D, Dinit=Dinit, mps_seed=cfg["seed"] + 1000, davidson_tol=1e-10, partial_bonds=nbonds,
                       sweeps=[dict(energy_last=r["energy_last"], energy_min=r["energy_min"],
                                    bonds=[dict(bond=b["bond"], dir=b["dir"], energy=b["energy"], kept=b["kept"],
                                                nsectors=b["nsectors"], trunc_err=b["trunc_err"], nnz=b["nnz"],
                                                n_matvec=b["n_matvec"]) for b in r["bonds"]]) for r in sweeps]),
                  f, indent=0)
    print(note, flush=True)


def golden_rdm(cid, D, nsample=0):
    """nsample > 0 (large k: Gamma has k^4 entries): store gamma, a seeded sample of nsample entries of Gamma (flat indices
    from default_rng(77)), and the full-array scalars sum Gamma^2 and sum_pr Gamma_pprr instead of Gamma itself."""
    cfg = make_config(cid)
    k, n = cfg["k"], cfg["n_elec"]
    mps = random_mps(k, n, cfg["two_sz"], D, seed=900 + cid, gauge="R")
    t0 = time.time()
    move = odmrg._move_centre_right

    def progress(m, c):                                     # progress line per centre (the pass takes hours at k = 54)
        print("  centre %d done, %.0f s" % (c, time.time() - t0), flush=True)
        return move(m, c)
    odmrg._move_centre_right = progress
    try:
        g, G = odmrg.rdm12(cfg["h"], cfg["eri"], mps, True)
    finally:
        odmrg._move_centre_right = move
    note = ("written by `python tests/golden/make_golden.py rdm %d %d%s` from oracle.dmrg.rdm12; oracle time %.0f s on "
            "%d host cores" % (cid, D, " %d" % nsample if nsample else "", time.time() - t0, os.cpu_count()))
    out = dict(gamma=g, D=D, config=cid, mps_seed=900 + cid, note=note)
    if nsample:
        idx = np.sort(np.random.default_rng(77).choice(G.size, size=nsample, replace=False))
        out.update(sample_idx=idx, sample_val=G.ravel()[idx], sum_sq=float(np.sum(G * G)),
                   trace2=float(np.einsum("pprr->", G)))
    else:
        out["Gamma"] = G
    np.savez_compressed(os.path.join(HERE, "rdm_cfg%d_D%d.npz" % (cid, D)), **out)
    print(note, flush=True)


def main():
    what = sys.argv[1] if len(sys.argv) > 1 else "fci"
    a = [int(x) for x in sys.argv[2:]]
    if what == "fci":
        golden_fci()
    elif what == "heff":
        golden_heff(a[0], a[1], a[2:])
    elif what == "sweep":
        golden_sweep(a[0], a[1], a[2], a[3] if len(a) > 3 else a[1], a[4] if len(a) > 4 else 0)
    elif what == "rdm":
        golden_rdm(a[0], a[1], a[2] if len(a) > 2 else 0)
    else:
        raise SystemExit(__doc__)


if __name__ == "__main__":
    main()
