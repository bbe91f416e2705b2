"""Generators for the five synthetic workloads of BASELINE.json (recipe: SURVEY.md section 8d).

They stand in for the paper's molecules / basis sets (branched alkanes + cc-pVTZ, water clusters,
transition-metal complexes + def2-TZVP), whose files are not available.
Everything is drawn from numpy.random.default_rng(240614920 + N); draw order: geometry, basis, density.
No integral / normalisation / screening arithmetic lives here.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

CONFIG_SEED = 240614920


def ncart(l: int) -> int:
    return (l + 1) * (l + 2) // 2


@dataclasses.dataclass
class Problem:
    """One J/K build problem.  Lengths in bohr; coefficients are RAW (un-normalised)."""

    name: str
    xyz: np.ndarray            # [natoms, 3] float64
    shell_atom: np.ndarray     # [nshells] int32
    shell_l: np.ndarray        # [nshells] int32, 0..3
    shell_nprim: np.ndarray    # [nshells] int32
    exponents: np.ndarray      # [sum nprim] float64, concatenated in shell order
    coefficients: np.ndarray   # [sum nprim] float64, raw contraction coefficients
    D: np.ndarray              # [nbf, nbf] float64 symmetric density, D = C C^T
    nocc: int
    tau_pair: float            # PQTHRE
    tau_jk: float              # THRECL

    @property
    def natoms(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def nshells(self) -> int:
        return int(self.shell_l.shape[0])

    @property
    def nbf(self) -> int:
        return int(sum(ncart(int(l)) for l in self.shell_l))

    @property
    def shell_offsets(self) -> np.ndarray:
        off = np.zeros(self.nshells + 1, dtype=np.int64)
        off[1:] = np.cumsum([ncart(int(l)) for l in self.shell_l])
        return off


# ----------------------------------------------------------------------------------------- geometry
def _unit(rng) -> np.ndarray:
    d = rng.normal(size=3)
    return d / np.linalg.norm(d)


def _chain(rng, n, start, others, lo=2.6, hi=2.9, minsp=2.6, box=None):
    """Self-avoiding random chain: step length uniform [lo,hi]; every non-neighbour (and every atom
    in `others`) at least `minsp` away; optional confinement to [0,box]^3."""
    pts = [np.asarray(start, dtype=float)]
    while len(pts) < n:
        for _ in range(100000):
            q = pts[-1] + _unit(rng) * rng.uniform(lo, hi)
            if box is not None and (np.any(q < 0.0) or np.any(q > box)):
                continue
            rest = pts[:-1] + list(others)
            if rest and np.min(np.linalg.norm(np.asarray(rest) - q, axis=1)) < minsp:
                continue
            pts.append(q)
            break
        else:  # pragma: no cover - never hit with these densities
            raise RuntimeError("self-avoiding chain stuck")
    return pts


def _add_h(rng, heavy, all_heavy, dist=2.05, min_heavy=2.6, min_h=2.0, tries=1000):
    """One H per heavy atom at `dist` in a random direction; rejected if within `min_heavy` of another
    heavy atom or `min_h` of another H (up to `tries` attempts, then the last try is kept)."""
    hs = []
    all_heavy = np.asarray(all_heavy)
    for h in heavy:
        q = None
        for _ in range(tries):
            q = h + dist * _unit(rng)
            dh = np.linalg.norm(all_heavy - q, axis=1)
            n_close = int(np.sum(dh < min_heavy))  # its own heavy atom is at 2.05 < 2.6
            if n_close > 1:
                continue
            if hs and np.min(np.linalg.norm(np.asarray(hs) - q, axis=1)) < min_h:
                continue
            break
        hs.append(q)
    return hs


# -------------------------------------------------------------------------------------------- basis
_R_ORG = {0: (0.05, 5000.0), 1: (0.1, 50.0), 2: (0.2, 5.0), 3: (0.4, 2.0)}
_HEAVY = {0: [6, 2, 1, 1, 1], 1: [4, 1, 1], 2: [1, 1], 3: [1]}
_HYD = {0: [3, 1, 1], 1: [1]}
_METAL = {0: [8, 3, 1, 1, 1, 1, 1], 1: [6, 2, 1, 1, 1], 2: [5, 1, 1, 1], 3: [1, 1]}
_R_MET = {l: (0.03, 1.0e5) for l in range(4)}


def _segmented_basis(rng, spec, ranges):
    """Per l: draw sum(lengths) log-uniform exponents, sort descending, cut into the contraction
    lengths in order (tightest -> most contracted shell); raw coefficients uniform [0.2, 1]."""
    shells = []
    for l, lengths in spec.items():
        lo, hi = ranges[l]
        ex = np.sort(np.exp(rng.uniform(math.log(lo), math.log(hi), sum(lengths))))[::-1]
        k = 0
        for c in lengths:
            shells.append((l, ex[k:k + c].copy(), rng.uniform(0.2, 1.0, c)))
            k += c
    return shells


def _assemble(name, atoms, rng, nocc, tau_pair, tau_jk) -> Problem:
    xyz = np.asarray([a[0] for a in atoms], dtype=np.float64).reshape(-1, 3)
    s_atom, s_l, s_np, ex, co = [], [], [], [], []
    for ia, (_, shells) in enumerate(atoms):
        for (l, e, c) in shells:
            s_atom.append(ia)
            s_l.append(l)
            s_np.append(len(e))
            ex.extend(e)
            co.extend(c)
    nbf = sum(ncart(l) for l in s_l)
    C = rng.normal(size=(nbf, nocc)) / math.sqrt(nbf)
    D = C @ C.T
    D = 0.5 * (D + D.T)
    return Problem(name=name, xyz=xyz,
                   shell_atom=np.asarray(s_atom, dtype=np.int32), shell_l=np.asarray(s_l, dtype=np.int32),
                   shell_nprim=np.asarray(s_np, dtype=np.int32),
                   exponents=np.asarray(ex, dtype=np.float64), coefficients=np.asarray(co, dtype=np.float64),
                   D=np.ascontiguousarray(D), nocc=nocc, tau_pair=tau_pair, tau_jk=tau_jk)


def make_config(n: int) -> Problem:
    """BASELINE.json configs[n-1], n = 1..5."""
    rng = np.random.default_rng(CONFIG_SEED + n)
    if n == 1:
        atoms = []
        pos = [rng.uniform(0.0, 6.0, 3) for _ in range(4)]
        for p in pos:
            shells = [(l, np.exp(rng.uniform(math.log(0.1), math.log(10.0), 3)), rng.uniform(0.2, 1.0, 3))
                      for l in range(4)]
            atoms.append((p, shells))
        return _assemble("cfg1_tiny", atoms, rng, nocc=10, tau_pair=0.0, tau_jk=0.0)
    if n == 2 or n == 5:
        nheavy = 12 if n == 2 else 120
        box = None if n == 2 else 40.0
        start = np.zeros(3) if n == 2 else np.full(3, 20.0)
        heavy = _chain(rng, nheavy, start, [], box=box)
        hs = _add_h(rng, heavy, heavy)
        bX = _segmented_basis(rng, _HEAVY, _R_ORG)
        bH = _segmented_basis(rng, _HYD, _R_ORG)
        atoms = [(p, bX) for p in heavy] + [(p, bH) for p in hs]
        name = "cfg2_small_organic" if n == 2 else "cfg5_large_organic"
        return _assemble(name, atoms, rng, nocc=40 if n == 2 else 480, tau_pair=1e-12, tau_jk=1e-12)
    if n == 3:
        th = math.radians(104.5)
        mols = []
        for ix in range(4):
            for iy in range(2):
                for iz in range(2):
                    O = 5.2 * np.array([ix, iy, iz], dtype=float) + rng.uniform(-0.3, 0.3, 3)
                    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
                    h1 = O + Q @ np.array([1.81, 0.0, 0.0])
                    h2 = O + Q @ np.array([1.81 * math.cos(th), 1.81 * math.sin(th), 0.0])
                    mols.append((O, h1, h2))
        bX = _segmented_basis(rng, _HEAVY, _R_ORG)
        bH = _segmented_basis(rng, _HYD, _R_ORG)
        atoms = []
        for (O, h1, h2) in mols:
            atoms += [(O, bX), (h1, bH), (h2, bH)]
        return _assemble("cfg3_water16", atoms, rng, nocc=80, tau_pair=1e-12, tau_jk=1e-12)
    if n == 4:
        # constructive reading of BASELINE.json: 6 chains x (8 heavy + 8 H) + metal = 97 atoms
        dirs = [np.array(v, dtype=float) for v in
                [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]]
        metal = np.zeros(3)
        heavy_all = []
        for d in dirs:
            st = d * rng.uniform(3.8, 4.2)
            heavy_all += _chain(rng, 8, st, [metal] + heavy_all)
        hs = _add_h(rng, heavy_all, [metal] + heavy_all)
        bM = _segmented_basis(rng, _METAL, _R_MET)
        bX = _segmented_basis(rng, _HEAVY, _R_ORG)
        bH = _segmented_basis(rng, _HYD, _R_ORG)
        atoms = [(metal, bM)] + [(p, bX) for p in heavy_all] + [(p, bH) for p in hs]
        return _assemble("cfg4_metal_complex", atoms, rng, nocc=230, tau_pair=1e-12, tau_jk=1e-12)
    raise ValueError("config number must be 1..5")


def digest(prob: Problem) -> dict:
    """SHA-256 of the generated arrays, so that "same inputs" can be checked across machines:
    `basis` covers geometry, shells, exponents and coefficients (pure functions of the seeded generator); `density`
    covers D = C C^T, whose last bits also depend on the BLAS that numpy calls for the product."""
    import hashlib
    hb, hd = hashlib.sha256(), hashlib.sha256()
    for a in (prob.xyz, prob.shell_atom, prob.shell_l, prob.shell_nprim, prob.exponents, prob.coefficients):
        hb.update(np.ascontiguousarray(a).tobytes())
    hd.update(np.ascontiguousarray(prob.D).tobytes())
    return {"basis": hb.hexdigest(), "density": hd.hexdigest()}


def subset_atoms(prob: Problem, atom_ids, name=None, max_l=None) -> Problem:
    """Cut-down problem: keep only the listed atoms (and optionally shells with l <= max_l); D is the
    matching principal sub-block (still symmetric PSD)."""
    atom_ids = [int(a) for a in atom_ids]
    remap = {a: i for i, a in enumerate(atom_ids)}
    off = prob.shell_offsets
    poff = np.zeros(prob.nshells + 1, dtype=np.int64)
    poff[1:] = np.cumsum(prob.shell_nprim)
    keep_sh = [s for a in atom_ids for s in range(prob.nshells)
               if int(prob.shell_atom[s]) == a and (max_l is None or int(prob.shell_l[s]) <= max_l)]
    ao = np.concatenate([np.arange(off[s], off[s + 1]) for s in keep_sh])
    pr = np.concatenate([np.arange(poff[s], poff[s + 1]) for s in keep_sh])
    return Problem(name=name or (prob.name + "_cut"), xyz=prob.xyz[atom_ids].copy(),
                   shell_atom=np.asarray([remap[int(prob.shell_atom[s])] for s in keep_sh], dtype=np.int32),
                   shell_l=prob.shell_l[keep_sh].copy(), shell_nprim=prob.shell_nprim[keep_sh].copy(),
                   exponents=prob.exponents[pr].copy(), coefficients=prob.coefficients[pr].copy(),
                   D=np.ascontiguousarray(prob.D[np.ix_(ao, ao)]), nocc=prob.nocc,
                   tau_pair=prob.tau_pair, tau_jk=prob.tau_jk)
