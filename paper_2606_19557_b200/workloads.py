"""Seeded synthetic workloads for the NEP training-step path (BASELINE.json configs 1-5).

This module serves BOTH the CPU oracle (tests) and the CUDA library (tests, bench, smoke).
It holds none of the method's arithmetic: only lattices, strains, displacements, species
draws and raw uniform draws for the parameter vector.  Anything that needs descriptors
(the scaler of Eq. 2; the centring of b0) is passed IN by the caller, who computes
it with whichever implementation is under test.

Recipe: SURVEY.md §8(d) / DESIGN.md "Input recipe".  The paper trains on published DFT
sets that are not available here; these synthetic sets stand in for them.

Determinism: root seed 260619557*10 + config_id, numpy PCG64; child streams are spawned
in a fixed order (structures, teacher, student, batches) and every structure draws from
its own grandchild stream, so the first k structures of a config are the same whether
k or the full count is requested.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional, Sequence, Tuple

import numpy as np

ROOT_SEED = 260619557 * 10


@dataclasses.dataclass(frozen=True)
class ModelSpec:
    """Hyper-parameters in the paper's input-file vocabulary (Table I)."""
    n_species: int
    rc_R: float
    rc_A: float
    n_max_R: int
    n_max_A: int
    basis_R: int
    basis_A: int
    l_max_3b: int = 4
    l_max_4b: int = 2
    l_max_5b: int = 1
    neurons: int = 30

    # inclusive ranges (pinned by Table II)
    @property
    def n_R(self) -> int:
        return self.n_max_R + 1

    @property
    def n_A(self) -> int:
        return self.n_max_A + 1

    @property
    def K_R(self) -> int:
        return self.basis_R + 1

    @property
    def K_A(self) -> int:
        return self.basis_A + 1

    @property
    def n_ang(self) -> int:
        return self.l_max_3b + (1 if self.l_max_4b > 0 else 0) + (1 if self.l_max_5b > 0 else 0)

    @property
    def D(self) -> int:
        return self.n_R + self.n_A * self.n_ang

    @property
    def n_par(self) -> int:
        T, H = self.n_species, self.neurons
        return T * (self.D + 2) * H + 1 + T * T * (self.n_R * self.K_R + self.n_A * self.K_A)

    def block_slices(self):
        """Flat theta layout (C0): per species w0[H*D], b0[H], w1[H]; b1; cR; cA."""
        T, H, D = self.n_species, self.neurons, self.D
        out = {}
        o = 0
        w0, b0, w1 = [], [], []
        for _ in range(T):
            w0.append(slice(o, o + H * D)); o += H * D
            b0.append(slice(o, o + H)); o += H
            w1.append(slice(o, o + H)); o += H
        out["w0"], out["b0"], out["w1"] = w0, b0, w1
        out["b1"] = slice(o, o + 1); o += 1
        n = T * T * self.n_R * self.K_R
        out["cR"] = slice(o, o + n); o += n
        n = T * T * self.n_A * self.K_A
        out["cA"] = slice(o, o + n); o += n
        assert o == self.n_par
        return out


@dataclasses.dataclass
class StructureSet:
    """Concatenated structures; Cartesian positions, rows of `box` are the cell vectors a, b, c."""
    n_atoms: np.ndarray   # [S] int32
    pos: np.ndarray       # [N,3] float64, wrapped to fractional [0,1)
    box: np.ndarray       # [S,9] float64 (rows a,b,c)
    type: np.ndarray      # [N] int32
    kind: List[str]       # [S] lattice tag, for reporting only

    @property
    def n_struct(self) -> int:
        return len(self.n_atoms)

    @property
    def atom_off(self) -> np.ndarray:
        return np.concatenate([[0], np.cumsum(self.n_atoms)]).astype(np.int64)

    def subset(self, ids: Sequence[int]) -> "StructureSet":
        off = self.atom_off
        idx = np.concatenate([np.arange(off[s], off[s + 1]) for s in ids]) if len(ids) else np.zeros(0, np.int64)
        return StructureSet(self.n_atoms[list(ids)].copy(), self.pos[idx].copy(), self.box[list(ids)].copy(),
                            self.type[idx].copy(), [self.kind[s] for s in ids])


@dataclasses.dataclass
class Workload:
    config_id: int
    name: str
    model: ModelSpec
    structures: StructureSet
    batch_size: int               # structures per step (BASELINE.json "batch")
    lambdas: Tuple[float, float, float]
    seeds: dict                   # name -> np.random.SeedSequence


# --------------------------------------------------------------------------------------
# lattices
# --------------------------------------------------------------------------------------
def _grid(nx, ny, nz):
    g = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij"), -1)
    return g.reshape(-1, 3).astype(np.float64)


def _lattice(kind: str, a: float, n: Tuple[int, int, int], c: float = 0.0):
    """Returns (positions [N,3], cell [3,3]) of an ideal supercell."""
    nx, ny, nz = n
    cells = _grid(nx, ny, nz)
    if kind == "fcc":
        basis = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]])
        unit = np.diag([a, a, a])
    elif kind == "bcc":
        basis = np.array([[0, 0, 0], [.5, .5, .5]])
        unit = np.diag([a, a, a])
    elif kind == "fcc_prim":
        basis = np.array([[0., 0, 0]])
        unit = 0.5 * a * np.array([[0, 1, 1], [1, 0, 1], [1, 1, 0]], float)
    elif kind == "hcp":  # orthohexagonal 4-atom cell (a, sqrt(3) a, c)
        basis = np.array([[0, 0, 0], [.5, .5, 0], [.5, 1. / 6., .5], [0, 2. / 3., .5]])
        unit = np.diag([a, math.sqrt(3.0) * a, c])
    else:
        raise ValueError(kind)
    frac = (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3)
    pos = frac @ unit
    cell = unit * np.array([[nx], [ny], [nz]], float)
    return pos, cell


def _wrap(pos, cell):
    """Wrap Cartesian positions so that fractional coordinates lie in [0,1)."""
    inv = np.linalg.inv(cell)
    f = pos @ inv
    f -= np.floor(f)
    f[f >= 1.0] = 0.0
    p = f @ cell
    # guard against f@cell landing a hair outside after rounding
    f2 = p @ inv
    bad = (f2 < 0.0) | (f2 >= 1.0)
    if bad.any():
        f[bad] = 0.0
        p = f @ cell
    return p


def _strain(rng, pos, cell, amp, diag=True):
    e = rng.uniform(-amp, amp, size=(3, 3))
    e = 0.5 * (e + e.T)
    if not diag:
        e[np.diag_indices(3)] = 0.0
    Fm = np.eye(3) + e
    return pos @ Fm.T, cell @ Fm.T


def _liquid(rng, N, density=0.08, dmin=1.8):
    """Random sequential insertion in a cubic periodic box with a minimum separation."""
    L = (N / density) ** (1.0 / 3.0)
    pts = np.zeros((N, 3))
    k = 0
    tries = 0
    while k < N:
        p = rng.uniform(0.0, L, size=3)
        tries += 1
        if k:
            d = pts[:k] - p
            d -= L * np.round(d / L)
            if (np.einsum("ij,ij->i", d, d) < dmin * dmin).any():
                if tries > 2000000:
                    raise RuntimeError("random sequential insertion did not converge")
                continue
        pts[k] = p
        k += 1
    return pts, np.eye(3) * L


# --------------------------------------------------------------------------------------
# per-config structure recipes; each takes the structure's own Generator
# --------------------------------------------------------------------------------------
def _s_cfg1(rng, variant):
    if variant == "1b":
        pos, cell = _lattice("fcc", 3.6, (4, 4, 4))
    else:
        pos, cell = _lattice("fcc_prim", 3.6, (4, 4, 4))
    pos = pos + rng.normal(scale=0.1, size=pos.shape)
    return pos, cell, np.zeros(len(pos), np.int32), "fcc"


def _s_cfg2(rng):
    pos, cell = _lattice("bcc", 3.16, (4, 4, 4))
    pos, cell = _strain(rng, pos, cell, 0.03)
    pos = pos + rng.normal(scale=0.15, size=pos.shape)
    return pos, cell, np.zeros(len(pos), np.int32), "bcc"


def _s_cfg3(rng):
    n = tuple(int(v) for v in rng.integers(3, 5, size=3))
    a = rng.uniform(3.6, 4.1)
    pos, cell = _lattice("fcc", a, n)
    pos, cell = _strain(rng, pos, cell, 0.05, diag=False)
    typ = rng.integers(0, 2, size=len(pos)).astype(np.int32)
    pos = pos + rng.normal(scale=0.2, size=pos.shape)
    if rng.uniform() < 0.05:
        k = int(rng.integers(0, len(pos)))
        pos = np.delete(pos, k, axis=0)
        typ = np.delete(typ, k)
    return pos, cell, typ, "fcc"


_BCC_SHAPES_4 = [(x, y, z) for x in range(4, 9) for y in range(4, 9) for z in range(4, 9)
                 if 128 <= 2 * x * y * z <= 512]


def _s_cfg4(rng):
    if rng.uniform() < 0.10:
        N = int(rng.integers(128, 513))
        pos, cell = _liquid(rng, N)
        kind = "liquid"
    else:
        n = _BCC_SHAPES_4[int(rng.integers(0, len(_BCC_SHAPES_4)))]
        pos, cell = _lattice("bcc", 3.16, n)
        pos, cell = _strain(rng, pos, cell, 0.03)
        pos = pos + rng.normal(scale=0.15, size=pos.shape)
        kind = "bcc"
    typ = rng.integers(0, 5, size=len(pos)).astype(np.int32)
    return pos, cell, typ, kind


def _closest_shape(per_cell, target, lo=32, hi=512):
    best = None
    for x in range(1, 9):
        for y in range(x, 9):
            for z in range(y, 9):
                cnt = per_cell * x * y * z
                if lo <= cnt <= hi:
                    key = (abs(cnt - target), z - x, cnt)
                    if best is None or key < best[0]:
                        best = (key, (x, y, z))
    return best[1]


def _s_cfg5(rng):
    target = int(round(32.0 * 16.0 ** rng.uniform()))
    target = min(max(target, 32), 512)
    lat = ("fcc", "bcc", "hcp", "random")[int(rng.integers(0, 4))]
    if lat == "random":
        pos, cell = _liquid(rng, target)
    else:
        per = {"fcc": 4, "bcc": 2, "hcp": 4}[lat]
        a = {"fcc": 3.6, "bcc": 3.16, "hcp": 2.95}[lat]
        shape = _closest_shape(per, target)
        shape = tuple(int(v) for v in rng.permutation(shape))
        pos, cell = _lattice(lat, a, shape, c=4.68)
        pos, cell = _strain(rng, pos, cell, 0.03)
        pos = pos + rng.normal(scale=0.15, size=pos.shape)
    typ = rng.integers(0, 4, size=len(pos)).astype(np.int32)
    return pos, cell, typ, lat


_CONFIGS = {
    1: dict(name="cfg1 fcc 1sp 8x64", n_struct=8, batch=8,
            model=ModelSpec(1, 5.0, 4.0, 4, 4, 8, 8, 4, 0, 0, 30)),
    2: dict(name="cfg2 bcc 1sp 1000x128", n_struct=1000, batch=1000,
            model=ModelSpec(1, 6.0, 4.0, 4, 4, 8, 8, 4, 2, 1, 30)),
    3: dict(name="cfg3 fcc alloy 2sp 2000x108-256", n_struct=2000, batch=500,
            model=ModelSpec(2, 6.0, 4.5, 6, 4, 10, 8, 4, 2, 1, 50)),
    4: dict(name="cfg4 bcc+liquid 5sp 4000x128-512", n_struct=4000, batch=1000,
            model=ModelSpec(5, 6.0, 4.0, 4, 4, 8, 8, 4, 2, 1, 30)),
    5: dict(name="cfg5 mixed 4sp 5000x32-512", n_struct=5000, batch=1000,
            model=ModelSpec(4, 6.0, 5.0, 4, 4, 8, 8, 4, 2, 1, 30)),
}


def config5_sweep() -> List[ModelSpec]:
    """The 8-point model-complexity sweep of config 5 (n_max x basis x neurons)."""
    out = []
    for nmax in (4, 8):
        for bas in (8, 12):
            for H in (30, 100):
                out.append(ModelSpec(4, 6.0, 5.0, nmax, nmax, bas, bas, 4, 2, 1, H))
    return out


def make_config(config_id: int, n_struct: Optional[int] = None, variant: str = "1a",
                model: Optional[ModelSpec] = None) -> Workload:
    """Build (a prefix of) BASELINE.json config `config_id` (1..5).

    n_struct: number of structures to generate (default: the config's full count).  The
    first k structures do not depend on k.  variant: "1a" (64-atom primitive-cell reading,
    primary) or "1b" (256-atom conventional-cell reading) for config 1.
    """
    cfg = _CONFIGS[config_id]
    S = cfg["n_struct"] if n_struct is None else int(n_struct)
    root = np.random.SeedSequence(ROOT_SEED + config_id)
    s_struct, s_teacher, s_student, s_batch = root.spawn(4)
    kids = s_struct.spawn(S)
    n_atoms, P, B, Ty, kinds = [], [], [], [], []
    for s in range(S):
        rng = np.random.Generator(np.random.PCG64(kids[s]))
        if config_id == 1:
            pos, cell, typ, kind = _s_cfg1(rng, variant)
        else:
            pos, cell, typ, kind = {2: _s_cfg2, 3: _s_cfg3, 4: _s_cfg4, 5: _s_cfg5}[config_id](rng)
        pos = _wrap(pos, cell)
        n_atoms.append(len(pos)); P.append(pos); B.append(cell.reshape(9)); Ty.append(typ); kinds.append(kind)
    st = StructureSet(np.asarray(n_atoms, np.int32), np.concatenate(P).astype(np.float64),
                      np.asarray(B, np.float64), np.concatenate(Ty).astype(np.int32), kinds)
    return Workload(config_id, cfg["name"], model or cfg["model"], st, min(cfg["batch"], S), (1.0, 1.0, 1.0),
                    dict(teacher=s_teacher, student=s_student, batch=s_batch))


# --------------------------------------------------------------------------------------
# parameter draws (paper silent on initialisation: DESIGN.md reading G19)
# --------------------------------------------------------------------------------------
class ParamDraw:
    """Two-phase draw of a flat parameter vector theta (float64).

    phase 1  coefficients(): cR, cA ~ U(-1,1)      -> caller computes descriptors q over the
                                                       set and the scaler s (Eq. 2) with them
    phase 2  network(qt_mean): w0 ~ U(-1,1)/sqrt(D); b0 = w0 . mean(q~) + U(-.5,.5);
                               w1 ~ U(-1,1); b1 ~ U(-1,1)
    `qt_mean` [D] is the mean over atoms of the SCALED descriptor, supplied by the caller.
    """

    def __init__(self, model: ModelSpec, seed: np.random.SeedSequence):
        self.model = model
        self.rng = np.random.Generator(np.random.PCG64(seed))
        self.theta = np.zeros(model.n_par, np.float64)
        self._phase = 0

    def coefficients(self) -> np.ndarray:
        assert self._phase == 0
        sl = self.model.block_slices()
        self.theta[sl["cR"]] = self.rng.uniform(-1.0, 1.0, size=sl["cR"].stop - sl["cR"].start)
        self.theta[sl["cA"]] = self.rng.uniform(-1.0, 1.0, size=sl["cA"].stop - sl["cA"].start)
        self._phase = 1
        return self.theta

    def network(self, qt_mean: np.ndarray) -> np.ndarray:
        assert self._phase == 1
        m = self.model
        sl = m.block_slices()
        qt_mean = np.asarray(qt_mean, np.float64).reshape(m.D)
        for t in range(m.n_species):
            w0 = self.rng.uniform(-1.0, 1.0, size=(m.neurons, m.D)) / math.sqrt(m.D)
            self.theta[sl["w0"][t]] = w0.reshape(-1)
            self.theta[sl["b0"][t]] = w0 @ qt_mean + self.rng.uniform(-0.5, 0.5, size=m.neurons)
            self.theta[sl["w1"][t]] = self.rng.uniform(-1.0, 1.0, size=m.neurons)
        self.theta[sl["b1"]] = self.rng.uniform(-1.0, 1.0, size=1)
        self._phase = 2
        return self.theta


def batches(workload: Workload) -> List[np.ndarray]:
    """Seeded permutation of structure ids cut into consecutive batches (last may be partial)."""
    S = workload.structures.n_struct
    rng = np.random.Generator(np.random.PCG64(workload.seeds["batch"]))
    perm = rng.permutation(S).astype(np.int32) if workload.batch_size < S else np.arange(S, dtype=np.int32)
    return [perm[i:i + workload.batch_size] for i in range(0, S, workload.batch_size)]


def tiny_workload(seed: int, n_species: int = 2, sizes: Sequence[int] = (5, 7), box: Sequence[float] = (3.4, 4.3),
                  model: Optional[ModelSpec] = None) -> Workload:
    """Very small random triclinic structures (boxes thinner than 2 rc: multi- and self-images).

    For oracle pins (finite differences) and for edge-case parity tests.
    """
    model = model or ModelSpec(n_species, 3.2, 2.6, 1, 1, 2, 2, 4, 2, 1, 4)
    root = np.random.SeedSequence(ROOT_SEED + 1000 + seed)
    s_struct, s_teacher, s_student, s_batch = root.spawn(4)
    rng = np.random.Generator(np.random.PCG64(s_struct))
    n_atoms, P, B, Ty = [], [], [], []
    for N, L in zip(sizes, box):
        cell = np.eye(3) * L + rng.normal(scale=0.2, size=(3, 3))
        if np.linalg.det(cell) < 0:
            cell[0] *= -1
        pos = rng.uniform(0.0, 1.0, size=(N, 3)) @ cell
        # keep atoms apart (>= 1.0 A incl. images) so finite differences stay smooth
        for _ in range(200):
            ok = True
            for i in range(N):
                for j in range(N):
                    for sh in np.ndindex(3, 3, 3):
                        if i == j and sh == (1, 1, 1):
                            continue
                        d = pos[j] - pos[i] + (np.array(sh) - 1) @ cell
                        if d @ d < 1.0:
                            pos[i] = rng.uniform(0.0, 1.0, size=3) @ cell
                            ok = False
            if ok:
                break
        pos = _wrap(pos, cell)
        n_atoms.append(N); P.append(pos); B.append(cell.reshape(9))
        Ty.append(rng.integers(0, model.n_species, size=N).astype(np.int32))
    st = StructureSet(np.asarray(n_atoms, np.int32), np.concatenate(P), np.asarray(B), np.concatenate(Ty),
                      ["tiny"] * len(n_atoms))
    return Workload(1000 + seed, f"tiny{seed}", model, st, len(n_atoms), (1.0, 2.0, 3.0),
                    dict(teacher=s_teacher, student=s_student, batch=s_batch))
