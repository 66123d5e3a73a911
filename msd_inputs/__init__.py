"""Seeded synthetic inputs for the MSD-AFQMC Wick's-theorem hot path.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2406_08314_b200/``).  It holds none of the method's arithmetic: it
draws random Hamiltonians, determinant lists, CI coefficients and walkers with
the shapes of BASELINE.json's five configs (which stand in for the paper's
[Cu2O2]2+ and [Fe2S2(SCH3)]2- workloads, PAPER.md:L303, L315 -- those integrals
and SCI trials are not available) and converts between the two equivalent
encodings of a determinant list (occupation lists <-> hole/particle tables).
Phases, overlaps, Green's functions etc. are computed separately by each side.

Recipe (readings A14-A18):
  draw order  h1, L, determinants, coefficients, walkers   from
  numpy.random.default_rng(seed).
"""
from __future__ import annotations

import dataclasses
import hashlib
from typing import Dict, Optional

import numpy as np

__all__ = ["CONFIGS", "MSDInputs", "generate", "occ_to_tables", "tables_to_occ",
           "near_reference_walkers", "walkers_from_rng", "wide_window"]


# name -> parameters.  "A" is the active-window size (orbitals around the Fermi
# level that excitations may touch); "level_law" selects how excitation levels
# are drawn (see _draw_levels); "coef_law" how CI coefficients are drawn.
CONFIGS: Dict[str, dict] = {
    # BASELINE.json configs[0]; reading A14: N_d = 36 binds.
    "tiny": dict(N=8, n_alpha=2, n_beta=2, n_chol=32, n_w=8, n_det=36, A=8,
                 level_law="tiny", max_level=2, coef_law="gauss_half",
                 chol_law="tiny", seed=0),
    # extra cheap cases named in reading A14
    "tiny-full": dict(N=8, n_alpha=2, n_beta=2, n_chol=32, n_w=8, n_det=199, A=8,
                      level_law="tiny", max_level=2, coef_law="gauss_half",
                      chol_law="tiny", seed=0),
    # BASELINE.json configs[1]
    "small": dict(N=32, n_alpha=8, n_beta=8, n_chol=200, n_w=64, n_det=1000, A=16,
                  level_law="uniform_total", max_level=4, coef_law="exp_level",
                  chol_law="norm_decay", seed=0),
    # BASELINE.json configs[2]
    "cu2o2": dict(N=80, n_alpha=16, n_beta=16, n_chol=600, n_w=200, n_det=10_000, A=24,
                  level_law="uniform_total", max_level=6, coef_law="loguniform",
                  coef_min=1e-6, chol_law="norm_decay", seed=0),
    # BASELINE.json configs[3]
    "fe2s2": dict(N=100, n_alpha=20, n_beta=20, n_chol=800, n_w=100, n_det=200_000, A=30,
                  level_law="binomial8", max_level=8, coef_law="loguniform",
                  coef_min=1e-7, chol_law="norm_decay", seed=0),
    # BASELINE.json configs[4]: one point of the sweep; n_det and max_level are
    # overridden by the caller (generate("sweep", n_det=..., max_level=...)).
    "sweep": dict(N=64, n_alpha=12, n_beta=12, n_chol=400, n_w=128, n_det=10_000, A=28,
                  level_law="uniform_per_spin", max_level=4, coef_law="loguniform",
                  coef_min=1e-6, chol_law="norm_decay", seed=0),
    # micro inputs for the Fock-space brute-force pins (2^(2N) amplitudes): not in BASELINE.json.
    "micro": dict(N=4, n_alpha=2, n_beta=1, n_chol=5, n_w=3, n_det=12, A=4,
                  level_law="uniform_total", max_level=3, coef_law="exp_level",
                  chol_law="norm_decay", seed=3, e0=0.7),
    "micro-cs": dict(N=5, n_alpha=2, n_beta=2, n_chol=6, n_w=2, n_det=40, A=5,
                     level_law="uniform_total", max_level=4, coef_law="gauss_half",
                     chol_law="tiny", seed=5, e0=-1.3),
    # open-shell case for n_alpha != n_beta (the paper's own example has
    # nocca=4, noccb=2: PAPER.md:L203-204); not in BASELINE.json.
    "open-shell": dict(N=12, n_alpha=4, n_beta=2, n_chol=24, n_w=6, n_det=150, A=10,
                       level_law="uniform_total", max_level=4, coef_law="exp_level",
                       chol_law="norm_decay", seed=0),
}


@dataclasses.dataclass
class MSDInputs:
    name: str
    N: int
    n_alpha: int
    n_beta: int
    n_chol: int
    n_w: int
    n_det: int
    e0: float
    h1: np.ndarray          # [N][N] f64 symmetric
    L: np.ndarray           # [n_chol][N][N] f64, each symmetric
    occ_ref_a: np.ndarray   # [n_alpha] int32 ascending
    occ_ref_b: np.ndarray   # [n_beta] int32 ascending
    occa: np.ndarray        # [n_det][n_alpha] int32 ascending occupation lists
    occb: np.ndarray        # [n_det][n_beta]
    exc_off_a: np.ndarray   # [n_det+1] int64 CSR offsets
    holes_a: np.ndarray     # int32, ascending within a determinant
    parts_a: np.ndarray
    exc_off_b: np.ndarray
    holes_b: np.ndarray
    parts_b: np.ndarray
    ci: np.ndarray          # [n_det] f64
    phi_a: np.ndarray       # [n_w][N][n_alpha] complex128
    phi_b: np.ndarray       # [n_w][N][n_beta]
    params: dict

    def sha256(self) -> str:
        h = hashlib.sha256()
        for a in (self.h1, self.L, self.occa, self.occb, self.ci, self.phi_a, self.phi_b):
            h.update(np.ascontiguousarray(a).tobytes())
        return h.hexdigest()

    def with_walkers(self, phi_a: np.ndarray, phi_b: np.ndarray) -> "MSDInputs":
        return dataclasses.replace(self, phi_a=np.ascontiguousarray(phi_a),
                                   phi_b=np.ascontiguousarray(phi_b), n_w=phi_a.shape[0])

    def subset_dets(self, idx) -> "MSDInputs":
        """Same inputs restricted to the determinants ``idx`` (order kept)."""
        idx = np.asarray(idx, dtype=np.int64)
        occa, occb = self.occa[idx], self.occb[idx]
        ta = occ_to_tables(occa, self.occ_ref_a)
        tb = occ_to_tables(occb, self.occ_ref_b)
        return dataclasses.replace(self, n_det=len(idx), occa=occa, occb=occb, ci=self.ci[idx].copy(),
                                   exc_off_a=ta[0], holes_a=ta[1], parts_a=ta[2],
                                   exc_off_b=tb[0], holes_b=tb[1], parts_b=tb[2])


# ----------------------------------------------------------------------------
# encodings
# ----------------------------------------------------------------------------
def wide_window(seed: int = 0, N: int = 116, n: int = 10, n_virt: int = 100, n_det: int = 600, max_level: int = 5,
                n_chol: int = 40, n_w: int = 9) -> "MSDInputs":
    """Closed-shell case whose active window is wider than the 16+16 orbitals of the BASELINE configs (the paper's
    [Cu2O2]2+ has 16 occupied x 92 virtual per spin): all n occupied orbitals and the lowest n_virt
    virtuals may be touched; total level uniform on 1..max_level, split binomially over the spins; reference first;
    coefficients |N(0,1)| exp(-level); h1, L and walkers as in generate("small")."""
    base = generate("small", seed=seed, N=N, n_alpha=n, n_beta=n, n_chol=n_chol, n_w=n_w, n_det=2, A=2 * min(n, 8))
    rng = np.random.default_rng(seed + 1000003)
    ref = np.arange(n, dtype=np.int32)
    rows, seen = [(tuple(ref), tuple(ref))], {(tuple(ref), tuple(ref))}
    while len(rows) < n_det:
        lev = int(rng.integers(1, max_level + 1))
        ka = int(rng.binomial(lev, 0.5))
        occ = []
        for k in (ka, lev - ka):
            k = min(k, n)
            keep = np.setdiff1d(ref, rng.choice(n, size=k, replace=False))
            occ.append(tuple(np.sort(np.concatenate([keep, n + rng.choice(n_virt, size=k, replace=False)])).tolist()))
        if tuple(occ) not in seen:
            seen.add(tuple(occ)); rows.append(tuple(occ))
    occa = np.array([r[0] for r in rows], dtype=np.int32)
    occb = np.array([r[1] for r in rows], dtype=np.int32)
    ta, tb = occ_to_tables(occa, ref), occ_to_tables(occb, ref)
    level = np.diff(ta[0]) + np.diff(tb[0])
    ci = np.abs(rng.standard_normal(n_det)) * np.exp(-1.0 * level)
    ci[0] = 1.0
    ci /= np.sqrt((ci * ci).sum())
    p = dict(base.params); p.update(n_det=n_det, max_level=max_level, wide_window=(n, n_virt))
    return dataclasses.replace(base, name="wide-window", n_det=n_det, occa=occa, occb=occb, ci=ci, params=p,
                               exc_off_a=ta[0], holes_a=ta[1], parts_a=ta[2], exc_off_b=tb[0], holes_b=tb[1], parts_b=tb[2])


def occ_to_tables(occ: np.ndarray, occ_ref: np.ndarray):
    """Occupation lists [n_det][n] -> CSR (off, holes, parts): holes = occ_ref \\ occ,
    parts = occ \\ occ_ref, both ascending.  Pure set bookkeeping."""
    occ = np.asarray(occ)
    n_det, n = occ.shape
    nmax = int(max(occ.max(initial=0), occ_ref.max(initial=0))) + 1 if n > 0 else 1
    in_ref = np.zeros(nmax, dtype=bool)
    in_ref[occ_ref] = True
    is_part = ~in_ref[occ]                                  # [n_det][n]
    k = is_part.sum(axis=1).astype(np.int64)
    off = np.zeros(n_det + 1, dtype=np.int64)
    np.cumsum(k, out=off[1:])
    parts = occ[is_part].astype(np.int32)                   # row-major: ascending inside each det
    occmask = np.zeros((n_det, nmax), dtype=bool)
    np.put_along_axis(occmask, occ.astype(np.int64), True, axis=1)
    hole_mask = ~occmask[:, occ_ref]                        # [n_det][n] in occ_ref order (ascending)
    holes = np.broadcast_to(occ_ref, (n_det, n))[hole_mask].astype(np.int32)
    return off, holes, parts


def tables_to_occ(off, holes, parts, occ_ref, n_det: int) -> np.ndarray:
    """Inverse of occ_to_tables: ascending occupation lists."""
    n = len(occ_ref)
    occ = np.empty((n_det, n), dtype=np.int32)
    for i in range(n_det):
        h = set(int(x) for x in holes[off[i]:off[i + 1]])
        o = [int(x) for x in occ_ref if int(x) not in h] + [int(x) for x in parts[off[i]:off[i + 1]]]
        occ[i] = sorted(o)
    return occ


# ----------------------------------------------------------------------------
# random pieces
# ----------------------------------------------------------------------------
def walkers_from_rng(rng: np.random.Generator, n_w: int, N: int, n: int) -> np.ndarray:
    """n_w random complex orthonormal N x n blocks: Q of the thin QR of a complex Gaussian."""
    out = np.empty((n_w, N, n), dtype=np.complex128)
    for w in range(n_w):
        z = rng.standard_normal((N, n)) + 1j * rng.standard_normal((N, n))
        q, _ = np.linalg.qr(z)
        out[w] = q
    return out


def near_reference_walkers(inp: "MSDInputs", eps: float, seed: int = 1, n_w: Optional[int] = None):
    """psi = QR(D_0 + eps * Z): what real AFQMC walkers look like (pin P8)."""
    rng = np.random.default_rng(seed)
    n_w = inp.n_w if n_w is None else n_w
    res = []
    for occ_ref, n in ((inp.occ_ref_a, inp.n_alpha), (inp.occ_ref_b, inp.n_beta)):
        out = np.empty((n_w, inp.N, n), dtype=np.complex128)
        for w in range(n_w):
            d0 = np.zeros((inp.N, n), dtype=np.complex128)
            d0[occ_ref, np.arange(n)] = 1.0
            z = rng.standard_normal((inp.N, n)) + 1j * rng.standard_normal((inp.N, n))
            q, _ = np.linalg.qr(d0 + eps * z)
            out[w] = q
        res.append(out)
    return res[0], res[1]


def _draw_levels(rng, law: str, max_level: int, m: int, kcap_a: int, kcap_b: int):
    """Per-spin excitation levels (ka, kb) for m candidate determinants (readings A15/A16)."""
    if law == "uniform_per_spin":            # config 5: iid uniform 0..K per spin, not both 0
        ka = rng.integers(0, max_level + 1, size=m)
        kb = rng.integers(0, max_level + 1, size=m)
    else:
        if law == "uniform_total":           # configs 2-3: total rank uniform on 1..lmax
            ell = rng.integers(1, max_level + 1, size=m)
        elif law == "binomial8":             # config 4: 1 + Binomial(7, 1/2): peaks at 4-5
            ell = 1 + rng.binomial(max_level - 1, 0.5, size=m)
        elif law == "tiny":                  # handled by enumeration, not here
            raise ValueError
        else:
            raise ValueError(law)
        ka = rng.binomial(ell, 0.5)
        kb = ell - ka
    ka = np.minimum(ka, kcap_a)
    kb = np.minimum(kb, kcap_b)
    keep = (ka + kb) > 0
    return ka[keep], kb[keep]


def _draw_subsets(rng, k: np.ndarray, universe: int) -> np.ndarray:
    """For each row i a uniformly random k[i]-subset of range(universe), as a bit mask (uint64)."""
    m = len(k)
    if universe == 0:
        return np.zeros(m, dtype=np.uint64)
    keys = rng.random((m, universe))
    order = np.argsort(keys, axis=1)                          # random permutation per row
    take = np.arange(universe)[None, :] < k[:, None]          # first k[i] entries of the permutation
    bits = (np.uint64(1) << order.astype(np.uint64)) * take.astype(np.uint64)
    return np.bitwise_or.reduce(bits, axis=1)


def _masks_to_occ(hmask, pmask, occ_ref, act_occ, act_virt):
    """Bit masks over the window -> ascending occupation lists."""
    m = len(hmask)
    n = len(occ_ref)
    nmax = int(max(occ_ref.max(initial=-1), act_virt.max(initial=-1))) + 1
    occm = np.zeros((m, nmax), dtype=bool)
    occm[:, occ_ref] = True
    for j, o in enumerate(act_occ):
        sel = ((hmask >> np.uint64(j)) & np.uint64(1)).astype(bool)
        occm[sel, o] = False
    for j, v in enumerate(act_virt):
        sel = ((pmask >> np.uint64(j)) & np.uint64(1)).astype(bool)
        occm[sel, v] = True
    # ascending orbital indices of the True entries, row by row
    cols = np.nonzero(occm)[1]
    return cols.reshape(m, n).astype(np.int32)


def _window(n: int, N: int, A: int):
    n_o = min(n, A // 2)
    n_v = min(A - n_o, N - n)
    act_occ = np.arange(n - n_o, n, dtype=np.int32)           # highest occupied
    act_virt = np.arange(n, n + n_v, dtype=np.int32)          # lowest virtual
    return act_occ, act_virt


def _tiny_determinants(rng, p, occ_ref_a, occ_ref_b, aoa, ava, aob, avb):
    """Reading A14: reference + (n_det-1) drawn without replacement from all non-reference
    determinants of total level <= max_level inside the window (198 of them for N=8, n=2)."""
    from itertools import combinations

    def strings(act_occ, act_virt):
        out = []
        for k in range(0, p["max_level"] + 1):
            for hs in combinations(range(len(act_occ)), k):
                for ps in combinations(range(len(act_virt)), k):
                    hm = sum(1 << j for j in hs)
                    pm = sum(1 << j for j in ps)
                    out.append((k, hm, pm))
        return out

    sa, sb = strings(aoa, ava), strings(aob, avb)
    allp = [(a, b) for a in sa for b in sb if 0 < a[0] + b[0] <= p["max_level"]]
    pick = rng.choice(len(allp), size=min(p["n_det"] - 1, len(allp)), replace=False)
    pick.sort()
    sel = [allp[i] for i in pick]
    hma = np.array([0] + [s[0][1] for s in sel], dtype=np.uint64)
    pma = np.array([0] + [s[0][2] for s in sel], dtype=np.uint64)
    hmb = np.array([0] + [s[1][1] for s in sel], dtype=np.uint64)
    pmb = np.array([0] + [s[1][2] for s in sel], dtype=np.uint64)
    return hma, pma, hmb, pmb


def generate(name: str, seed: Optional[int] = None, **overrides) -> MSDInputs:
    """Generate one config.  ``overrides`` may change any parameter (n_det, n_w, max_level, ...)."""
    p = dict(CONFIGS[name])
    p.update(overrides)
    if seed is not None:
        p["seed"] = seed
    rng = np.random.default_rng(p["seed"])
    N, na, nb, ng, nw, nd = p["N"], p["n_alpha"], p["n_beta"], p["n_chol"], p["n_w"], p["n_det"]

    # --- h1 ---------------------------------------------------------------
    a = rng.standard_normal((N, N))
    h1 = 0.5 * (a + a.T)

    # --- L (reading A17) ----------------------------------------------------
    a = rng.standard_normal((ng, N, N))
    s = 0.5 * (a + a.transpose(0, 2, 1))
    if p["chol_law"] == "tiny":
        L = s * np.exp(-np.arange(ng) / 8.0)[:, None, None]
    else:
        tau = p.get("chol_tau", ng / 5.0)
        nrm = np.sqrt((s * s).sum(axis=(1, 2)))
        L = s / nrm[:, None, None] * np.exp(-np.arange(ng) / tau)[:, None, None]
    del a, s

    # --- determinants -------------------------------------------------------
    occ_ref_a = np.arange(na, dtype=np.int32)
    occ_ref_b = np.arange(nb, dtype=np.int32)
    aoa, ava = _window(na, N, p["A"])
    aob, avb = _window(nb, N, p["A"])
    kcap_a = min(len(aoa), len(ava))
    kcap_b = min(len(aob), len(avb))
    if p["level_law"] == "tiny":
        hma, pma, hmb, pmb = _tiny_determinants(rng, p, occ_ref_a, occ_ref_b, aoa, ava, aob, avb)
        nd = len(hma)
    else:
        nva, nvb = len(ava), len(avb)
        keys_seen = np.zeros(1, dtype=np.uint64)              # the reference: all masks 0
        rows = [np.zeros((1, 4), dtype=np.uint64)]
        have = 1
        guard = 0
        while have < nd:
            m = int((nd - have) * 1.3) + 64
            ka, kb = _draw_levels(rng, p["level_law"], p["max_level"], m, kcap_a, kcap_b)
            ha = _draw_subsets(rng, ka, len(aoa))
            pa = _draw_subsets(rng, ka, nva)
            hb = _draw_subsets(rng, kb, len(aob))
            pb = _draw_subsets(rng, kb, nvb)
            # 64-bit key; windows are <= 16+16 per spin in every config (asserted)
            assert len(aoa) <= 16 and nva <= 16 and len(aob) <= 16 and nvb <= 16
            key = (ha | (pa << np.uint64(16)) | (hb << np.uint64(32)) | (pb << np.uint64(48)))
            # first occurrence inside the batch, and not seen before; keep draw order
            _, first = np.unique(key, return_index=True)
            first.sort()
            key = key[first]
            fresh = ~np.isin(key, keys_seen)
            sel = first[fresh][: nd - have]
            rows.append(np.stack([ha[sel], pa[sel], hb[sel], pb[sel]], axis=1))
            keys_seen = np.concatenate([keys_seen, key[fresh][: nd - have]])
            have += len(sel)
            guard += 1
            if guard > 200:
                raise RuntimeError("determinant space exhausted: lower n_det or raise max_level")
        allrows = np.concatenate(rows, axis=0)
        hma, pma, hmb, pmb = (allrows[:, j].copy() for j in range(4))
    occa = _masks_to_occ(hma, pma, occ_ref_a, aoa, ava)
    occb = _masks_to_occ(hmb, pmb, occ_ref_b, aob, avb)
    ta = occ_to_tables(occa, occ_ref_a)
    tb = occ_to_tables(occb, occ_ref_b)
    level = (ta[0][1:] - ta[0][:-1]) + (tb[0][1:] - tb[0][:-1])

    # --- coefficients -------------------------------------------------------
    law = p["coef_law"]
    if law == "gauss_half":
        ci = rng.standard_normal(nd) * np.exp(-0.5 * level)
    elif law == "exp_level":
        ci = np.abs(rng.standard_normal(nd)) * np.exp(-1.0 * level)
    elif law == "loguniform":
        lo = np.log(p["coef_min"])
        ci = np.exp(rng.uniform(lo, 0.0, size=nd)) * rng.choice([-1.0, 1.0], size=nd)
    else:
        raise ValueError(law)
    ci[0] = 1.0
    ci = ci / np.sqrt((ci * ci).sum())

    # --- walkers ------------------------------------------------------------
    phi_a = walkers_from_rng(rng, nw, N, na)
    phi_b = walkers_from_rng(rng, nw, N, nb)

    p["n_det"] = nd
    return MSDInputs(name=name, N=N, n_alpha=na, n_beta=nb, n_chol=ng, n_w=nw, n_det=nd,
                     e0=float(p.get("e0", 0.0)), h1=h1, L=np.ascontiguousarray(L),
                     occ_ref_a=occ_ref_a, occ_ref_b=occ_ref_b, occa=occa, occb=occb,
                     exc_off_a=ta[0], holes_a=ta[1], parts_a=ta[2],
                     exc_off_b=tb[0], holes_b=tb[1], parts_b=tb[2],
                     ci=ci, phi_a=phi_a, phi_b=phi_b, params=p)
