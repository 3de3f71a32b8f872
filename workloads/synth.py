"""Seeded synthetic inputs shaped like the paper's workloads (harness, not product).

This module holds NONE of the method's arithmetic: no scoring, kinematics, pair lists,
RNG-for-the-chains.  It only builds the INPUT arrays that the fp64 oracle (``oracle/``)
and the CUDA library (``paper_2510_24186_b200``) both consume, so that the two never
have to share code.  Recipe: SURVEY.md section 8(d) / DESIGN.md section 4; configs C1..C5
are BASELINE.json ``configs[0..4]``.

The paper's own inputs (PDBbind time-split complexes, DEKOIS 2.0 targets, PAPER.md
lines 75-79, 270, 297) are not available offline; these seeded receptors/ligands
stand in for them with the same shapes (pocket-sized receptor, drug-like ligands,
AutoDock-style 0.375 A grid).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "_ligand_gen.so")
_SRC = os.path.join(_HERE, "ligand_gen.c")


def build(force: bool = False) -> str:
    """Compile the ligand generator (plain C, gcc)."""
    import hashlib
    want = hashlib.sha256(open(_SRC, "rb").read()).hexdigest()
    stamp = _SO + ".stamp"
    if force or not os.path.exists(_SO) or not os.path.exists(stamp) or open(stamp).read() != want:
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"])
        with open(stamp, "w") as f:
            f.write(want)
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.ligand_gen_batch.restype = ctypes.c_int
    return _lib


# ----------------------------------------------------------------------------- types
def type_table(n_types: int):
    """Synthetic atom-type table (the paper takes vdW radii and H-bond
    roles from OpenBabel and never lists them).

    radius[t] = 1.5 + 0.1*(t mod 8) + 0.05*(t div 8)  [A];
    hb_role[t mod 8] = {0,0,1,2,0,0,3,0}  (bit0 donor, bit1 acceptor)."""
    t = np.arange(n_types)
    radius = (1.5 + 0.1 * (t % 8) + 0.05 * (t // 8)).astype(np.float32)
    role = np.array([0, 0, 1, 2, 0, 0, 3, 0], dtype=np.uint8)[t % 8]
    return radius, role


# -------------------------------------------------------------------------- receptor
@dataclass
class Receptor:
    xyz: np.ndarray          # [n_rec,3] float32
    type: np.ndarray         # [n_rec] int32
    n_types: int
    box_len: float
    origin: np.ndarray       # [3] float32, grid origin (cube corner)
    dims: tuple              # (nx, ny, nz)
    spacing: float
    pocket_center: np.ndarray
    pocket_radius: float
    box_min: np.ndarray
    box_max: np.ndarray
    min_sep: float


def receptor(n_rec: int, box_len: float, n_types: int, seed: int, grid_n: int,
             pocket_radius: float = 8.0, spacing: float = 0.375) -> Receptor:
    """Random sequential addition of n_rec points uniform in [0,L]^3 outside the central
    pocket sphere, min separation s = min(3 A, 0.8*(V_free/n_rec)^(1/3)) (BASELINE.json's
    literal 3 A jams before n_rec atoms are placed -- SURVEY 8(d))."""
    rng = np.random.default_rng(seed)
    centre = np.full(3, box_len / 2.0)
    v_free = box_len ** 3 - 4.0 / 3.0 * np.pi * pocket_radius ** 3
    s = min(3.0, 0.8 * (v_free / n_rec) ** (1.0 / 3.0))
    ncell = max(1, int(box_len / s))
    cell = box_len / ncell
    cells: dict = {}
    pts = np.empty((n_rec, 3))
    n = 0
    trials = 0
    while n < n_rec:
        batch = rng.uniform(0.0, box_len, size=(4096, 3))
        for p in batch:
            trials += 1
            if np.sum((p - centre) ** 2) < pocket_radius ** 2:
                continue
            ci = tuple(np.minimum((p / cell).astype(int), ncell - 1))
            ok = True
            for dx in (-1, 0, 1):
                for dy in (-1, 0, 1):
                    for dz in (-1, 0, 1):
                        for j in cells.get((ci[0] + dx, ci[1] + dy, ci[2] + dz), ()):
                            if np.sum((pts[j] - p) ** 2) < s * s:
                                ok = False
                                break
                        if not ok:
                            break
                    if not ok:
                        break
                if not ok:
                    break
            if not ok:
                continue
            pts[n] = p
            cells.setdefault(ci, []).append(n)
            n += 1
            if n == n_rec:
                break
        if trials > 4_000_000:
            raise RuntimeError("receptor RSA did not converge")
    types = rng.integers(0, n_types, size=n_rec).astype(np.int32)
    return Receptor(
        xyz=pts.astype(np.float32), type=types, n_types=n_types, box_len=box_len,
        origin=np.zeros(3, np.float32), dims=(grid_n, grid_n, grid_n), spacing=spacing,
        pocket_center=centre.astype(np.float32), pocket_radius=pocket_radius,
        box_min=(centre - pocket_radius).astype(np.float32),
        box_max=(centre + pocket_radius).astype(np.float32), min_sep=s)


# --------------------------------------------------------------------------- ligands
@dataclass
class LigandBatch:
    """CSR-packed ligand batch, exactly the arrays of ``tridsk_ligand_batch`` (include/tridsk.h)."""
    n_lig: int
    atom_off: np.ndarray     # [n_lig+1] int32
    ref_xyz: np.ndarray      # [sum n,3] float32, centred on the centroid
    atom_type: np.ndarray    # [sum n] uint8
    atom_frag: np.ndarray    # [sum n] uint8   0 = root fragment, k+1 = child fragment of torsion k
    tor_off: np.ndarray      # [n_lig+1] int32
    tor_a: np.ndarray        # [sum T] uint8   axis a->b, a on the root side
    tor_b: np.ndarray        # [sum T] uint8
    tor_parent: np.ndarray   # [sum T] int8    -1 = root; parents precede children
    bond_off: np.ndarray     # [n_lig+1] int32
    bond_ab: np.ndarray      # [sum nb,2] uint8

    def n_atoms(self, i):
        return int(self.atom_off[i + 1] - self.atom_off[i])

    def n_tor(self, i):
        return int(self.tor_off[i + 1] - self.tor_off[i])

    def one(self, i) -> dict:
        """Arrays of ligand i (views)."""
        a0, a1 = self.atom_off[i], self.atom_off[i + 1]
        t0, t1 = self.tor_off[i], self.tor_off[i + 1]
        b0, b1 = self.bond_off[i], self.bond_off[i + 1]
        return dict(ref_xyz=self.ref_xyz[a0:a1], atom_type=self.atom_type[a0:a1],
                    atom_frag=self.atom_frag[a0:a1], tor_a=self.tor_a[t0:t1],
                    tor_b=self.tor_b[t0:t1], tor_parent=self.tor_parent[t0:t1],
                    bond_ab=self.bond_ab[b0:b1])

    def subset(self, idx) -> "LigandBatch":
        idx = list(idx)
        parts = [self.one(i) for i in idx]
        cat = lambda k, dt, shp: (np.concatenate([p[k] for p in parts]).astype(dt)
                                  if parts else np.zeros(shp, dt))
        off = lambda k: np.concatenate([[0], np.cumsum([len(p[k]) for p in parts])]).astype(np.int32)
        return LigandBatch(
            n_lig=len(idx), atom_off=off("atom_type"), ref_xyz=cat("ref_xyz", np.float32, (0, 3)),
            atom_type=cat("atom_type", np.uint8, (0,)), atom_frag=cat("atom_frag", np.uint8, (0,)),
            tor_off=off("tor_a"), tor_a=cat("tor_a", np.uint8, (0,)), tor_b=cat("tor_b", np.uint8, (0,)),
            tor_parent=cat("tor_parent", np.int8, (0,)), bond_off=off("bond_ab"),
            bond_ab=cat("bond_ab", np.uint8, (0, 2)))


def ligands(n_atoms, n_tor_req, n_types: int, seed: int, backbone: int = 0) -> LigandBatch:
    """Grow len(n_atoms) tree ligands (see ligand_gen.c for the recipe)."""
    lib = _load()
    n = np.ascontiguousarray(n_atoms, dtype=np.int32)
    tr = np.ascontiguousarray(n_tor_req, dtype=np.int32)
    L = len(n)
    atom_off = np.concatenate([[0], np.cumsum(n)]).astype(np.int32)
    cap_off = np.concatenate([[0], np.cumsum(tr)]).astype(np.int32)
    tot, cap = int(atom_off[-1]), int(cap_off[-1])
    xyz = np.zeros((tot, 3), np.float32)
    typ = np.zeros(tot, np.uint8)
    frag = np.zeros(tot, np.uint8)
    bonds = np.zeros((max(tot - L, 0), 2), np.uint8)
    ta = np.zeros(max(cap, 1), np.uint8)
    tb = np.zeros(max(cap, 1), np.uint8)
    tp = np.zeros(max(cap, 1), np.int8)
    t_out = np.zeros(L, np.int32)
    P = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    rc = lib.ligand_gen_batch(ctypes.c_uint64(seed), ctypes.c_int(L), P(n), P(tr), ctypes.c_int(n_types),
                              ctypes.c_int(backbone), P(atom_off), P(cap_off), P(xyz), P(typ), P(bonds),
                              P(frag), P(ta), P(tb), P(tp), P(t_out))
    if rc != 0:
        raise RuntimeError("ligand generator failed")
    # compact the torsion arrays from capacity offsets to actual counts
    tor_off = np.concatenate([[0], np.cumsum(t_out)]).astype(np.int32)
    sel = np.zeros(max(cap, 1), bool)
    for_idx = np.repeat(cap_off[:-1], t_out) + (np.arange(int(tor_off[-1])) - np.repeat(tor_off[:-1], t_out))
    sel[for_idx] = True
    bond_off = (atom_off - np.arange(L + 1)).astype(np.int32)
    return LigandBatch(n_lig=L, atom_off=atom_off, ref_xyz=xyz, atom_type=typ, atom_frag=frag,
                       tor_off=tor_off, tor_a=ta[sel].copy(), tor_b=tb[sel].copy(), tor_parent=tp[sel].copy(),
                       bond_off=bond_off, bond_ab=bonds)


# --------------------------------------------------------------------------- configs
@dataclass
class Config:
    name: str
    title: str
    n_rec: int
    box_len: float
    grid_n: int
    n_types: int
    n_lig: int
    n_chains: int
    n_steps: int
    top_k: int
    rec_seed: int
    lig_seed: int
    philox_seed: int = 0
    backbone: int = 0
    sizes: dict = field(default_factory=dict)
    n_refine: int = 1
    direct: bool = False         # the receptor term by direct pair sums instead of the grid lookup (S:8(f) NEXT-3)
    mdn_K: int = 0               # > 0: the workload carries the mixture-density term with K components per (residue, atom)


CONFIGS = {
    "C1": Config("C1", "Tiny", 300, 20.0, 54, 8, 1, 64, 100, 1, 1001, 2001),
    "C2": Config("C2", "Drug-like single dock", 3000, 30.0, 80, 16, 1, 384, 1000, 10, 1002, 2002),
    "C3": Config("C3", "Screening batch", 3000, 30.0, 80, 16, 4096, 128, 500, 1, 1003, 2003),
    "C4": Config("C4", "Large flexible ligand", 3000, 40.0, 107, 16, 1, 1024, 2000, 1, 1004, 2004, backbone=24),
    "C5": Config("C5", "High-throughput screen", 5000, 30.0, 80, 16, 65536, 64, 300, 1, 1005, 2005),
    # Not a BASELINE.json config: the sampling shape the paper states for its own runs (1,024 copies, depth 8,
    # Adam refinement in every loop; 8 output poses) on the C2 receptor and ligand.  The number of Adam iterations
    # per loop is not stated in the paper; 32 is this build's choice (G12).
    # Not a BASELINE.json config: 32 independent copies of the C2 dock in one batch ("C2 run as 32 concurrent
    # independent docks to show the kernel's rate when fed")
    "C2x32": Config("C2x32", "32 concurrent drug-like single docks", 3000, 30.0, 80, 16, 32, 384, 1000, 10, 1002, 2002),
    # Not a BASELINE.json config: the first 1,024 ligands of C3 sampled under the paper's FULL score, E_MDN included (SURVEY
    # 8(f) NEXT-1), with synthetic mixture parameters (K = 10) on the pocket residues (pocket_residues below).
    "M3": Config("M3", "Screening batch under the full score (E_MDN, K = 10), first 1,024 ligands of C3", 3000, 30.0, 80, 16, 1024, 128, 500, 1,
                 1003, 2003, mdn_K=10),
    # Not a BASELINE.json config: the C2 dock under the paper's FULL score (E_MDN, K = 10, pocket residues): the paper's own use
    # case for "ms per docking task"
    "M2": Config("M2", "Drug-like single dock under the full score (E_MDN, K = 10)", 3000, 30.0, 80, 16, 1, 384, 1000, 10, 1002, 2002,
                 mdn_K=10),
    # Not a BASELINE.json config: C2 docked with the receptor term taken the paper's own way, direct sums over the receptor atoms
    # within the pair function's range, 200 MC steps
    "D2": Config("D2", "Drug-like single dock, receptor term by direct pair sums", 3000, 30.0, 80, 16, 1, 384, 200, 10, 1002, 2002, direct=True),
    "P1": Config("P1", "Paper-shaped run (1,024 copies x 8 loops x 32 Adam steps)", 3000, 30.0, 80, 16, 1, 1024, 8, 8, 1002, 2002,
                 n_refine=32),
}


def config_sizes(cfg: Config, n_lig: int | None = None):
    """Per-ligand (n_atoms, n_tor_requested) arrays for a config (BASELINE.json configs)."""
    L = cfg.n_lig if n_lig is None else n_lig
    rng = np.random.default_rng(cfg.lig_seed)
    if cfg.name == "C1":
        return np.full(L, 12), np.full(L, 2)
    if cfg.name in ("C2", "P1", "C2x32", "D2", "M2"):
        return np.full(L, 30), np.full(L, 6)
    if cfg.name in ("C3", "M3"):
        n = rng.integers(15, 51, size=4096)
        t = np.array([rng.integers(0, min(12, k // 4) + 1) for k in n])
        return n[:L], t[:L]                                                  # ligand i is the same in C3 and M3
    if cfg.name == "C4":
        return np.full(L, 80), np.full(L, 20)
    if cfg.name == "C5":
        n = np.clip(np.rint(rng.normal(28.0, 8.0, size=cfg.n_lig)), 10, 70).astype(int)
        t = np.minimum(rng.poisson(5.0, size=cfg.n_lig), 15)
        return n[:L], t[:L]
    raise KeyError(cfg.name)


def make_receptor(cfg: Config) -> Receptor:
    return receptor(cfg.n_rec, cfg.box_len, cfg.n_types, cfg.rec_seed, cfg.grid_n)


def make_ligands(cfg: Config, n_lig: int | None = None) -> LigandBatch:
    """First n_lig ligands of the config (ligand i is the same whatever n_lig is)."""
    n, t = config_sizes(cfg, n_lig)
    return ligands(n, t, cfg.n_types, cfg.lig_seed, backbone=cfg.backbone)


def random_poses(batch: LigandBatch, lig_index, rec: Receptor, seed: int, spread: float = 1.0):
    """Random test poses [n_pose, 7+Tmax] float32: translation uniform in the search box
    (scaled by `spread` about the pocket centre), uniform unit quaternion, torsions uniform."""
    rng = np.random.default_rng(seed)
    lig_index = np.asarray(lig_index, dtype=np.int32)
    tmax = int(np.max(np.diff(batch.tor_off))) if batch.n_lig else 0
    n = len(lig_index)
    poses = np.zeros((n, 7 + tmax), np.float32)
    half = (rec.box_max - rec.box_min) / 2 * spread
    poses[:, 0:3] = rec.pocket_center + rng.uniform(-1, 1, size=(n, 3)) * half
    q = rng.normal(size=(n, 4))
    poses[:, 3:7] = q / np.linalg.norm(q, axis=1, keepdims=True)
    poses[:, 7:] = rng.uniform(-np.pi, np.pi, size=(n, tmax))
    for i, li in enumerate(lig_index):
        poses[i, 7 + batch.n_tor(li):] = 0.0
    return poses


# --------------------------------------------------------------------------- fixed waters
def with_waters(rec: "Receptor", n_water: int, seed: int, water_type: int = 6, min_sep: float = 2.6):
    """The receptor with n_water crystallographic-style waters kept as FIXED receptor atoms (Tables S8/S9 P:567-629):
    oxygen positions drawn uniformly in the shell 1 A inside the pocket wall, at least min_sep from every receptor atom and
    from one another; type `water_type` (donor + acceptor in the synthetic table).  -> a new Receptor (same grid geometry)."""
    rng = np.random.default_rng(seed)
    xyz, typ = [r for r in rec.xyz], list(rec.type)
    placed, tries = 0, 0
    while placed < n_water and tries < 200000:
        tries += 1
        v = rng.normal(size=3)
        v /= np.linalg.norm(v)
        p = rec.pocket_center + v * rng.uniform(rec.pocket_radius - 2.0, rec.pocket_radius - 0.5)
        if np.min(np.linalg.norm(np.asarray(xyz) - p, axis=1)) < min_sep:
            continue
        xyz.append(p.astype(np.float32)); typ.append(water_type); placed += 1
    out = Receptor(**{**rec.__dict__})
    out.xyz = np.asarray(xyz, np.float32)
    out.type = np.asarray(typ, np.int32)
    return out


# --------------------------------------------------------------------------- inputs of E_MDN
def residues(rec: "Receptor", size: int = 8):
    """Group the receptor atoms into spatially compact pseudo-residues of `size` atoms (the paper's residues come from
    the protein's sequence, which a synthetic point cloud does not have): atoms are ordered by the Morton code of their
    5 A cell and cut into consecutive groups.  -> (order [n_rec] permutation of the atoms, res_off [n_res+1])."""
    cell = np.floor((rec.xyz - rec.xyz.min(axis=0)) / 5.0).astype(np.int64)
    code = np.zeros(len(cell), np.int64)
    for b in range(6):
        for c in range(3):
            code |= ((cell[:, c] >> b) & 1) << (3 * b + c)
    order = np.lexsort((np.arange(len(code)), code))
    n_res = (len(order) + size - 1) // size
    res_off = np.minimum(np.arange(n_res + 1) * size, len(order)).astype(np.int32)
    return order, res_off


def pocket_residues(rec: "Receptor", size: int = 8, reach: float = 13.0):
    """The residues E_MDN runs over: the paper uses the POCKET residues (those near the ligand); here the groups of
    `size` receptor atoms (residues above) that have an atom within `reach` of the pocket centre (search box 8 A + the 5 A
    cut-off of the term).  -> (res_xyz [n_at,3] float32, res_off [n_res+1] int32)."""
    order, off = residues(rec, size)
    xyz = rec.xyz[order]
    keep_xyz, keep_off = [], [0]
    for i in range(len(off) - 1):
        a = xyz[off[i]:off[i + 1]]
        if len(a) and np.min(np.linalg.norm(a - rec.pocket_center, axis=1)) < reach:
            keep_xyz.append(a)
            keep_off.append(keep_off[-1] + len(a))
    return np.concatenate(keep_xyz).astype(np.float32), np.asarray(keep_off, np.int32)


def gmm_batch(n_res: int, n_atoms, K: int, seed: int):
    """gmm_params for every ligand of a batch, flat and ligand-major (the layout tridsk_load_mdn takes):
    -> pi, mu, sigma float32 [sum_l n_res * n_atoms[l] * K]."""
    out = [[], [], []]
    for l, n in enumerate(n_atoms):
        for dst, a in zip(out, gmm_params(n_res, int(n), K, seed + l)):
            dst.append(a.reshape(-1))
    return tuple(np.concatenate(v) for v in out)


def gmm_params(n_res: int, n_atoms: int, K: int, seed: int):
    """Synthetic mixture parameters standing in for the graph transformer's output (trained weights are not
    here): pi ~ Dirichlet(1) over K, mu ~ U(2.5, 6.0) A, sigma ~ U(0.3, 1.2) A.  -> pi, mu, sigma float32 [n_res][n_atoms][K]."""
    rng = np.random.default_rng(seed)
    pi = rng.dirichlet(np.ones(K), size=(n_res, n_atoms)).astype(np.float32)
    mu = rng.uniform(2.5, 6.0, size=(n_res, n_atoms, K)).astype(np.float32)
    sigma = rng.uniform(0.3, 1.2, size=(n_res, n_atoms, K)).astype(np.float32)
    return pi, mu, sigma
