"""ctypes shim over oracle/tridsk_oracle.c -- the plain fp64 CPU oracle.

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs may import this.  It never imports the CUDA package and shares no
code with it.  Argument marshalling only; every number is computed in tridsk_oracle.c, except
O13 (top-k = a lexicographic sort, done here with numpy.lexsort) and E_screen.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tridsk_oracle.c")
_SO = os.path.join(_HERE, "_tridsk_oracle.so")


def build(force: bool = False) -> str:
    """gcc -O2, no -ffast-math."""
    import hashlib
    want = hashlib.sha256(open(_SRC, "rb").read()).hexdigest()
    stamp = _SO + ".stamp"
    if force or not os.path.exists(_SO) or not os.path.exists(stamp) or open(stamp).read() != want:
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"])
        with open(stamp, "w") as f:
            f.write(want)
    return _SO


class Params(C.Structure):
    _fields_ = [(n, C.c_double) for n in (
        "w_long", "w_clash", "w_hbond", "long_mu", "long_two_sigma2", "long_dmax",
        "hb_mu", "hb_sigma", "hb_dmax", "hb_dclash", "d_floor", "k_wall",
        "beta", "lr", "adam_b1", "adam_b2", "adam_eps", "pert_trans", "pert_rot", "w_tor")] + [
        ("n_refine", C.c_int), ("clash_literal", C.c_int)]


class _Types(C.Structure):
    _fields_ = [("n_types", C.c_int), ("radius", C.c_void_p), ("role", C.c_void_p)]


class _Grid(C.Structure):
    _fields_ = [("g", C.c_void_p), ("n_types", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("origin", C.c_double * 3), ("spacing", C.c_double), ("rec_xyz", C.c_void_p), ("rec_type", C.c_void_p),
                ("n_rec", C.c_int)]


class _Mdn(C.Structure):
    _fields_ = [("n_res", C.c_int), ("K", C.c_int), ("res_off", C.c_void_p), ("res_xyz", C.c_void_p), ("pi", C.c_void_p),
                ("mu", C.c_void_p), ("sigma", C.c_void_p), ("w_mdn", C.c_double), ("d_cut", C.c_double)]


class _Ligand(C.Structure):
    _fields_ = [("n", C.c_int), ("T", C.c_int), ("P", C.c_int), ("ref", C.c_void_p), ("type", C.c_void_p),
                ("frag", C.c_void_p), ("tor_a", C.c_void_p), ("tor_b", C.c_void_p), ("tor_parent", C.c_void_p),
                ("pairs", C.c_void_p), ("mdn", C.c_void_p)]


class StepRec(C.Structure):
    _fields_ = [("e_prop", C.c_double), ("e_cur", C.c_double), ("u", C.c_double), ("accept", C.c_int),
                ("entity", C.c_int), ("min_abs_g", C.c_double), ("p_accept", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_field_brute.restype = C.c_double
        _lib.orc_derive_pairs.restype = C.c_int
        assert _lib.orc_sizeof_params() == C.sizeof(Params)
        assert _lib.orc_sizeof_step_rec() == C.sizeof(StepRec)
        assert _lib.orc_sizeof_ligand() == C.sizeof(_Ligand) and _lib.orc_sizeof_mdn() == C.sizeof(_Mdn)
        assert _lib.orc_sizeof_grid() == C.sizeof(_Grid)
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _d3(v):
    return (C.c_double * 3)(*[float(x) for x in v])


def default_params(**kw) -> Params:
    p = Params()
    lib().orc_default_params(C.byref(p))
    for k, v in kw.items():
        setattr(p, k, v)
    return p


class Types:
    def __init__(self, radius, role):
        self.radius = np.ascontiguousarray(radius, dtype=np.float64)
        self.role = np.ascontiguousarray(role, dtype=np.uint8)
        self.c = _Types(len(self.radius), _p(self.radius).value, _p(self.role).value)


class Grid:
    """Wraps an fp32 [n_types][nz][ny][nx] array (O4); the hot-path oracle reads it as handed."""

    def __init__(self, g, origin, spacing):
        self.g = np.ascontiguousarray(g, dtype=np.float32)
        nt, nz, ny, nx = self.g.shape
        self.origin = np.asarray(origin, dtype=np.float64)
        self.spacing = float(spacing)
        self.c = _Grid(_p(self.g).value, nt, nx, ny, nz, _d3(origin), float(spacing), None, None, 0)


class DirectReceptor:
    """Stands where a Grid stands in score_grad / mc_step / dock, but makes the receptor term the paper's own direct sums over
    the receptor atoms (P:103-125, P:353 item 4): no grid, no interpolation, no wall."""

    def __init__(self, rec_xyz, rec_type, n_types):
        self.xyz = np.ascontiguousarray(rec_xyz, dtype=np.float64)
        self.type = np.ascontiguousarray(rec_type, dtype=np.int32)
        self.g = np.zeros((n_types, 2, 2, 2), np.float32)
        self.c = _Grid(_p(self.g).value, n_types, 2, 2, 2, _d3([0, 0, 0]), 1.0, _p(self.xyz).value, _p(self.type).value, len(self.type))


class Ligand:
    def __init__(self, ref_xyz, atom_type, atom_frag, tor_a, tor_b, tor_parent, bond_ab=None, pairs=None):
        self.ref = np.ascontiguousarray(ref_xyz, dtype=np.float64)
        self.type = np.ascontiguousarray(atom_type, dtype=np.uint8)
        self.frag = np.ascontiguousarray(atom_frag, dtype=np.uint8)
        self.tor_a = np.ascontiguousarray(tor_a, dtype=np.uint8)
        self.tor_b = np.ascontiguousarray(tor_b, dtype=np.uint8)
        self.tor_parent = np.ascontiguousarray(tor_parent, dtype=np.int8)
        self.n, self.T = len(self.type), len(self.tor_a)
        if pairs is None:
            pairs = derive_pairs(self.frag, bond_ab)
        self.pairs = np.ascontiguousarray(pairs, dtype=np.uint8).reshape(-1, 2)
        self.P = len(self.pairs)
        self.c = _Ligand(self.n, self.T, self.P, _p(self.ref).value, _p(self.type).value, _p(self.frag).value,
                         _p(self.tor_a).value, _p(self.tor_b).value, _p(self.tor_parent).value,
                         _p(self.pairs).value, None)
        self.mdn = None

    def set_mdn(self, mdn: "Mdn | None"):
        """Attach (or detach, None) the mixture-density term: every score / MC step of this ligand then uses the paper's
        full E_dock = w_MDN E_MDN + w_long E_long + w_clash E_clash + w_Hbond E_Hbond."""
        if mdn is not None:
            assert mdn.pi.shape[1] == self.n
        self.mdn = mdn
        self.c.mdn = C.addressof(mdn.c) if mdn is not None else None
        return self


class Mdn:
    """O15 inputs for ONE ligand: residues of the receptor (res_off into res_xyz) and the mixture parameters
    pi, mu, sigma [n_res][n_atoms][K] of every (residue, ligand atom) pair (Eq.GMM)."""

    def __init__(self, res_xyz, res_off, pi, mu, sigma, w_mdn=1.0, d_cut=5.0):
        self.res_xyz = np.ascontiguousarray(res_xyz, dtype=np.float64)
        self.res_off = np.ascontiguousarray(res_off, dtype=np.int32)
        self.pi, self.mu, self.sigma = (np.ascontiguousarray(a, dtype=np.float64) for a in (pi, mu, sigma))
        n_res, n, K = self.pi.shape
        assert len(self.res_off) == n_res + 1 and self.mu.shape == self.pi.shape == self.sigma.shape
        self.c = _Mdn(n_res, K, _p(self.res_off).value, _p(self.res_xyz).value, _p(self.pi).value, _p(self.mu).value,
                      _p(self.sigma).value, float(w_mdn), float(d_cut))


def mdn_energy(res_xyz, res_off, pi, mu, sigma, x, d_cut=5.0):
    """orc_mdn_energy (O15): -> (E_MDN, dE/dx [n][3], d [n_res][n]).  Same signature as oracle.mdn.mdn_energy."""
    M = Mdn(res_xyz, res_off, pi, mu, sigma, 1.0, d_cut)
    x = np.ascontiguousarray(x, dtype=np.float64)
    n = x.shape[0]
    e = C.c_double()
    g = np.zeros((n, 3))
    dm = np.zeros((M.c.n_res, n))
    lib().orc_mdn_energy(C.byref(M.c), C.c_int(n), _p(x), C.byref(e), _p(g), _p(dm))
    return float(e.value), g, dm


def ligand_from_batch(batch, i) -> Ligand:
    """batch: workloads.synth.LigandBatch (plain arrays)."""
    d = batch.one(i)
    return Ligand(d["ref_xyz"], d["atom_type"], d["atom_frag"], d["tor_a"], d["tor_b"], d["tor_parent"],
                  bond_ab=d["bond_ab"])


# ------------------------------------------------------------------------------ O2..O5
def pair(p: Params, rad_s, role_s, rad_t, role_t, d):
    e, de = C.c_double(), C.c_double()
    lib().orc_pair(C.byref(p), C.c_double(rad_s), C.c_ubyte(role_s), C.c_double(rad_t), C.c_ubyte(role_t),
                   C.c_double(d), C.byref(e), C.byref(de))
    return e.value, de.value


def field_brute(p, ty: Types, rec_xyz, rec_type, t, x):
    rx = np.ascontiguousarray(rec_xyz, dtype=np.float64)
    rt = np.ascontiguousarray(rec_type, dtype=np.int32)
    return lib().orc_field_brute(C.byref(p), C.byref(ty.c), _p(rx), _p(rt), C.c_int(len(rt)), C.c_int(t), _d3(x))


def build_grid(p, ty: Types, rec_xyz, rec_type, origin, dims, spacing) -> Grid:
    rx = np.ascontiguousarray(rec_xyz, dtype=np.float64)
    rt = np.ascontiguousarray(rec_type, dtype=np.int32)
    nx, ny, nz = dims
    out = np.zeros((ty.c.n_types, nz, ny, nx), np.float32)
    lib().orc_build_grid(C.byref(p), C.byref(ty.c), _p(rx), _p(rt), C.c_int(len(rt)), _d3(origin),
                         C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(spacing), _p(out))
    return Grid(out, origin, spacing)


def interp(p, G: Grid, t, x):
    e = C.c_double()
    g = (C.c_double * 3)()
    lib().orc_interp(C.byref(p), C.byref(G.c), C.c_int(t), _d3(x), C.byref(e), g)
    return e.value, np.array(g[:])


# ------------------------------------------------------------------------------ O6, O8, O9
def derive_pairs(frag, bond_ab):
    frag = np.ascontiguousarray(frag, dtype=np.uint8)
    bonds = np.ascontiguousarray(bond_ab, dtype=np.uint8).reshape(-1, 2)
    n = len(frag)
    cap = n * (n - 1) // 2 + 1
    out = np.zeros((cap, 2), np.uint8)
    P = lib().orc_derive_pairs(C.c_int(n), _p(frag), _p(bonds), C.c_int(len(bonds)), _p(out), C.c_int(cap))
    return out[:P].copy()


def fk(L: Ligand, pose):
    pose = np.ascontiguousarray(pose, dtype=np.float64)
    x = np.zeros((L.n, 3))
    lib().orc_fk(C.byref(L.c), _p(pose), _p(x))
    return x


def score_grad(p, ty: Types, G: Grid, L: Ligand, pose, want_grad=True):
    """-> energy[3] (total, inter, intra), grad[6+T], coords[n,3], gatom[n,3]."""
    pose = np.ascontiguousarray(pose, dtype=np.float64)
    e = np.zeros(3)
    g = np.zeros(6 + L.T)
    x = np.zeros((L.n, 3))
    ga = np.zeros((L.n, 3))
    lib().orc_score_grad(C.byref(p), C.byref(ty.c), C.byref(G.c), C.byref(L.c), _p(pose), _p(e),
                         _p(g) if want_grad else None, _p(x), _p(ga))
    return e, g, x, ga


def score_grad_direct(p, ty: Types, rec_xyz, rec_type, L: Ligand, pose, want_grad=True):
    """The same evaluation with the receptor term as the paper's direct sums over receptor atoms (no grid, no wall;
    SURVEY 8(f) NEXT-3).  -> energy[3], grad[6+T], coords[n,3], gatom[n,3]."""
    pose = np.ascontiguousarray(pose, dtype=np.float64)
    xyz = np.ascontiguousarray(rec_xyz, dtype=np.float64)
    typ = np.ascontiguousarray(rec_type, dtype=np.int32)
    e = np.zeros(3)
    g = np.zeros(6 + L.T)
    x = np.zeros((L.n, 3))
    ga = np.zeros((L.n, 3))
    lib().orc_score_grad_direct(C.byref(p), C.byref(ty.c), _p(xyz), typ.ctypes.data_as(C.c_void_p), C.c_int(len(typ)),
                                C.byref(L.c), _p(pose), _p(e), _p(g) if want_grad else None, _p(x), _p(ga))
    return e, g, x, ga


def score_grad_batch(p, ty: Types, G: Grid, L: Ligand, poses):
    poses = np.ascontiguousarray(poses, dtype=np.float64)
    n, stride = poses.shape
    e = np.zeros((n, 3))
    g = np.zeros((n, 6 + L.T))
    x = np.zeros((n, L.n, 3))
    lib().orc_score_grad_batch(C.byref(p), C.byref(ty.c), C.byref(G.c), C.byref(L.c), _p(poses), C.c_int(n),
                               C.c_int(stride), _p(e), _p(g), C.c_int(6 + L.T), _p(x), C.c_int(L.n))
    return e, g, x


# ------------------------------------------------------------------------------ O10..O12
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return list(o)


def uniform4(seed, chain, step, ligand, purpose):
    u = (C.c_double * 4)()
    lib().orc_uniform4(C.c_uint64(seed), C.c_uint32(chain), C.c_uint32(step), C.c_uint32(ligand),
                       C.c_uint32(purpose), u)
    return np.array(u[:])


def init_pose(L: Ligand, seed, chain, ligand, centre, radius):
    pose = np.zeros(7 + L.T)
    lib().orc_init_pose(C.byref(L.c), C.c_uint64(seed), C.c_uint32(chain), C.c_uint32(ligand), _d3(centre),
                        C.c_double(radius), _p(pose))
    return pose


def mc_step(p, ty, G, L, seed, chain, step, ligand, box_min, box_max, pose, e_cur):
    """One MC step from (pose, e_cur).  -> new pose, new e_cur, StepRec."""
    pose = np.array(pose, dtype=np.float64)
    ec = C.c_double(e_cur)
    rec = StepRec()
    lib().orc_mc_step(C.byref(p), C.byref(ty.c), C.byref(G.c), C.byref(L.c), C.c_uint64(seed), C.c_uint32(chain),
                      C.c_uint32(step), C.c_uint32(ligand), _d3(box_min), _d3(box_max), _p(pose), C.byref(ec),
                      C.byref(rec))
    return pose, ec.value, rec


def dock(p, ty, G, L, seed, ligand, n_chains, n_steps, box_min, box_max, centre, radius,
         init_poses=None, first_step=0, want_trace=False):
    W = 7 + L.T
    ip = None
    if init_poses is not None:
        ip = np.ascontiguousarray(np.asarray(init_poses, dtype=np.float64)[:, :W])
        assert ip.shape == (n_chains, W)
    e_best = np.zeros(n_chains)
    e_cur = np.zeros(n_chains)
    pose_best = np.zeros((n_chains, W))
    pose_cur = np.zeros((n_chains, W))
    trace = (StepRec * (n_chains * n_steps))() if want_trace else None
    lib().orc_dock(C.byref(p), C.byref(ty.c), C.byref(G.c), C.byref(L.c), C.c_uint64(seed), C.c_uint32(ligand),
                   C.c_int(n_chains), C.c_int(first_step), C.c_int(n_steps), _d3(box_min), _d3(box_max),
                   _d3(centre), C.c_double(radius), _p(ip) if ip is not None else None, C.c_int(W),
                   _p(e_best), _p(pose_best), _p(e_cur), _p(pose_cur), trace)
    out = dict(e_best=e_best, pose_best=pose_best, e_cur=e_cur, pose_cur=pose_cur)
    if want_trace:
        names = [f[0] for f in StepRec._fields_]
        out["trace"] = {n: np.array([getattr(r, n) for r in trace]).reshape(n_chains, n_steps) for n in names}
    return out


# ------------------------------------------------------------------------------ O13, E_screen
def topk(e_best, k):
    """O13: chains sorted by (E_best, chain id) ascending, first k."""
    e_best = np.asarray(e_best)
    order = np.lexsort((np.arange(len(e_best)), e_best))
    return order[:k]


def topk_cluster(e_best, pose_best, L: Ligand, k, rmsd_min):
    """O14 ("ranked ... clustered to remove the duplicates ... top N"; reading G20): walk the chains in the order
    of O13; a chain's best pose is a duplicate if its heavy-atom RMSD (same atom order, no superposition: poses live in
    the receptor frame) to an already kept pose is below rmsd_min, otherwise it is kept; stop at k kept.
    -> (kept chain ids, length <= k; margin = the smallest |RMSD - rmsd_min| met on the way, for tie detection)."""
    e_best = np.asarray(e_best)
    order = np.lexsort((np.arange(len(e_best)), e_best))
    kept, kept_x, margin = [], [], np.inf
    for c in order:
        if len(kept) == k:
            break
        x = fk(L, np.asarray(pose_best[c], dtype=np.float64)[:7 + L.T])
        dup = False
        for kx in kept_x:                                     # plain loop, in kept order; every comparison is made
            rmsd = float(np.sqrt(np.mean(np.sum((x - kx) ** 2, axis=1))))
            margin = min(margin, abs(rmsd - rmsd_min))
            if rmsd < rmsd_min:
                dup = True
                break
        if not dup:
            kept.append(int(c))
            kept_x.append(x)
    return np.array(kept, dtype=np.int64), margin


def e_screen(e_dock, n_tor, w_tor=0.01):
    """Eq.E_screen."""
    return e_dock / (1.0 + w_tor * n_tor)
