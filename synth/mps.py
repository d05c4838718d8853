"""Seeded block-sparse random MPS in the neutral exchange format.

Input generation only.  Format (plain Python containers, host memory):
  mps["bonds"][b]   for b = 0..k : list of (N, two_sz, dim), sorted ascending by (N, two_sz); bond 0 = [(0,0,1)],
                    bond k = [(n_elec, two_sz, 1)]   (Eq. 14: boundary bonds of dimension 1)
  mps["tensors"][p] for p = 0..k-1: dict {(l_idx, s): float64 array [dim_l, dim_r]} for every left sector l_idx of
                    bond p and site state s in {0: empty, 1: down, 2: up, 3: up-down} whose right
                    sector q_l + q(s) exists on bond p+1
  mps["gauge"][p]   "L" (left-orthonormal), "R" (right-orthonormal) or "C".
"""
import numpy as np

SITE_Q = ((0, 0), (1, -1), (1, 1), (2, 0))      # (N, 2Sz) of |0>, |dn>, |up>, |up dn>


def _count_tables(k):
    """cnt[b][(N, S2)] = number of product states of b sites with quantum numbers (N, S2)."""
    cnt = [{(0, 0): 1}]
    for _ in range(k):
        nxt = {}
        for (n, s), c in cnt[-1].items():
            for (dn, ds) in SITE_Q:
                key = (n + dn, s + ds)
                nxt[key] = nxt.get(key, 0) + c
        cnt.append(nxt)
    return cnt


def full_sector_dims(k, n_elec, two_sz):
    """Exact Schmidt-rank bound per bond and sector: d_full(b, q) = min(#left states(q), #right states(target-q))."""
    cnt = _count_tables(k)
    out = []
    for b in range(k + 1):
        d = {}
        for (n, s), cl in cnt[b].items():
            cr = cnt[k - b].get((n_elec - n, two_sz - s), 0)
            if cr > 0:
                d[(n, s)] = min(cl, cr)
        out.append(d)
    return out


def bond_sector_plan(k, n_elec, two_sz, D, sigma_n=1.6, sigma_s=2.2, min_dim=1):
    """Choose sector dimensions for every bond: weights Gaussian around the mean filling N*b/k and 2Sz*b/k,
    scaled to sum ~D, capped by d_full, then clipped until an isometry exists in both gauges
    (d_r <= sum_{(l,s)->r} d_l and d_l <= sum_{(s,r)<-l} d_r).  Returns list over bonds of {(N,S2): dim}."""
    full = full_sector_dims(k, n_elec, two_sz)
    plan = []
    for b in range(k + 1):
        tot_full = sum(full[b].values())
        if tot_full <= D:
            plan.append(dict(full[b]))
            continue
        nbar = n_elec * b / k
        sbar = two_sz * b / k
        keys = sorted(full[b].keys())
        w = np.array([np.exp(-0.5 * ((n - nbar) / sigma_n) ** 2 - 0.5 * ((s - sbar) / sigma_s) ** 2)
                      for (n, s) in keys])
        w = w / w.sum()
        d = {}
        for key, wi in zip(keys, w):
            v = int(round(D * wi))
            v = min(v, full[b][key])
            if v >= min_dim:
                d[key] = v
        plan.append(d)
    for _ in range(4 * k):
        changed = False
        for b in range(k):                                    # left-isometry feasibility on bond b+1
            for (n, s) in list(plan[b + 1].keys()):
                cap = sum(plan[b].get((n - dn, s - ds), 0) for (dn, ds) in SITE_Q)
                if plan[b + 1][(n, s)] > cap:
                    changed = True
                    if cap > 0:
                        plan[b + 1][(n, s)] = cap
                    else:
                        del plan[b + 1][(n, s)]
        for b in range(k - 1, -1, -1):                        # right-isometry feasibility on bond b
            for (n, s) in list(plan[b].keys()):
                cap = sum(plan[b + 1].get((n + dn, s + ds), 0) for (dn, ds) in SITE_Q)
                if plan[b][(n, s)] > cap:
                    changed = True
                    if cap > 0:
                        plan[b][(n, s)] = cap
                    else:
                        del plan[b][(n, s)]
        if not changed:
            break
    return plan


def _orth_rows(rng, rows, cols):
    """Random [rows, cols] matrix with orthonormal rows (rows <= cols)."""
    m = rng.normal(size=(cols, rows))
    q, r = np.linalg.qr(m)
    q = q * np.sign(np.diag(r))[None, :]
    return np.ascontiguousarray(q.T)


def random_mps(k, n_elec, two_sz, D, seed, gauge="R", plan=None):
    """Seeded random block-sparse MPS with N(0,1)-then-orthonormalised tensors.
    gauge "R": every site right-orthonormal (sum_s B[s] B[s]^T = 1 per left sector);
    gauge "L": every site left-orthonormal (sum_s A[s]^T A[s] = 1 per right sector);
    gauge "LR:i": sites < i left-orthonormal, sites >= i right-orthonormal ("dual gauge" for H_eff at bond i).
    Sites are generated in index order, sectors/blocks in sorted order, so the stream is reproducible."""
    rng = np.random.default_rng(seed)
    if plan is None:
        plan = bond_sector_plan(k, n_elec, two_sz, D)
    bonds = [sorted((n, s, d) for (n, s), d in plan[b].items()) for b in range(k + 1)]
    index = [{(n, s): i for i, (n, s, d) in enumerate(bonds[b])} for b in range(k + 1)]
    if gauge.startswith("LR:"):
        split = int(gauge[3:])
        gl = ["L" if p < split else "R" for p in range(k)]
    else:
        gl = [gauge] * k
    tensors = []
    for p in range(k):
        T = {}
        if gl[p] == "R":
            for li, (n, s, dl) in enumerate(bonds[p]):
                outs = [(st, index[p + 1][(n + dn, s + ds)]) for st, (dn, ds) in enumerate(SITE_Q)
                        if (n + dn, s + ds) in index[p + 1]]
                widths = [bonds[p + 1][ri][2] for (_, ri) in outs]
                tot = sum(widths)
                assert tot >= dl, "sector plan does not admit a right isometry"
                M = _orth_rows(rng, dl, tot)
                off = 0
                for (st, ri), wdt in zip(outs, widths):
                    T[(li, st)] = np.ascontiguousarray(M[:, off:off + wdt])
                    off += wdt
        else:
            for ri, (n, s, dr) in enumerate(bonds[p + 1]):
                ins = [(index[p][(n - dn, s - ds)], st) for st, (dn, ds) in enumerate(SITE_Q)
                       if (n - dn, s - ds) in index[p]]
                ins.sort()
                heights = [bonds[p][li][2] for (li, _) in ins]
                tot = sum(heights)
                assert tot >= dr, "sector plan does not admit a left isometry"
                M = _orth_rows(rng, dr, tot).T                      # [tot, dr] orthonormal columns
                off = 0
                for (li, st), hgt in zip(ins, heights):
                    T[(li, st)] = np.ascontiguousarray(M[off:off + hgt, :])
                    off += hgt
        tensors.append(T)
    return dict(k=k, n_elec=n_elec, two_sz=two_sz, bonds=bonds, tensors=tensors, gauge=gl)


def dual_gauge_mps(k, n_elec, two_sz, D, seed):
    """A left-orthonormal MPS A (seed) and a right-orthonormal MPS B (seed + 1) on ONE sector plan: H_eff at any
    two-site bond i is defined by A on sites < i and B on sites > i + 1, so one pair serves every bond."""
    plan = bond_sector_plan(k, n_elec, two_sz, D)
    A = random_mps(k, n_elec, two_sz, D, seed=seed, gauge="L", plan=plan)
    B = random_mps(k, n_elec, two_sz, D, seed=seed + 1, gauge="R", plan=plan)
    return A, B


def mixed_gauge(A, B, i):
    """Sites < i from A (left-orthonormal), sites >= i from B (right-orthonormal); same bonds."""
    k = A["k"]
    assert A["bonds"] == B["bonds"]
    return dict(k=k, n_elec=A["n_elec"], two_sz=A["two_sz"], bonds=A["bonds"],
                tensors=[A["tensors"][p] if p < i else B["tensors"][p] for p in range(k)],
                gauge=["L" if p < i else "R" for p in range(k)])


def mps_to_blob_arrays(mps):
    """Flatten to the C-ABI blob: (bond_ptr[k+2], sec_N, sec_S2, sec_dim, blk_ptr[k+1], blk_l, blk_s, blk_off, data,
    gauge bytes).  Blocks of a site are ordered by (l_idx, s); offsets are in doubles into `data`."""
    k = mps["k"]
    bond_ptr = [0]
    sn, ss, sd = [], [], []
    for b in range(k + 1):
        for (n, s, d) in mps["bonds"][b]:
            sn.append(n), ss.append(s), sd.append(d)
        bond_ptr.append(len(sn))
    blk_ptr = [0]
    bl, bs, bo = [], [], []
    chunks = []
    off = 0
    for p in range(k):
        for (li, st) in sorted(mps["tensors"][p].keys()):
            a = mps["tensors"][p][(li, st)]
            bl.append(li), bs.append(st), bo.append(off)
            chunks.append(np.ascontiguousarray(a, dtype=np.float64).ravel())
            off += a.size
        blk_ptr.append(len(bl))
    data = np.concatenate(chunks) if chunks else np.zeros(0)
    gauge = np.frombuffer("".join(mps["gauge"]).encode(), dtype=np.uint8).copy()
    return (np.array(bond_ptr, dtype=np.int32), np.array(sn, dtype=np.int32), np.array(ss, dtype=np.int32),
            np.array(sd, dtype=np.int32), np.array(blk_ptr, dtype=np.int32), np.array(bl, dtype=np.int32),
            np.array(bs, dtype=np.int32), np.array(bo, dtype=np.int64), data, gauge)


def blob_arrays_to_mps(k, n_elec, two_sz, bond_ptr, sn, ss, sd, blk_ptr, bl, bs, bo, data, gauge):
    """Inverse of mps_to_blob_arrays."""
    bonds = [[(int(sn[i]), int(ss[i]), int(sd[i])) for i in range(bond_ptr[b], bond_ptr[b + 1])]
             for b in range(k + 1)]
    index = [{(n, s): i for i, (n, s, d) in enumerate(bonds[b])} for b in range(k + 1)]
    tensors = []
    for p in range(k):
        T = {}
        for j in range(blk_ptr[p], blk_ptr[p + 1]):
            li, st = int(bl[j]), int(bs[j])
            n, s, dl = bonds[p][li]
            ri = index[p + 1][(n + SITE_Q[st][0], s + SITE_Q[st][1])]
            dr = bonds[p + 1][ri][2]
            T[(li, st)] = np.array(data[bo[j]:bo[j] + dl * dr]).reshape(dl, dr)
        tensors.append(T)
    return dict(k=k, n_elec=n_elec, two_sz=two_sz, bonds=bonds, tensors=tensors,
                gauge=[chr(c) for c in gauge])
