"""Pins for the fp64 oracle (oracle/) against what the paper and the mathematics fix.

None of these retypes the oracle's own formula: each is a printed constant, a closed form at a
special point, an invariant, a library routine (scipy / torch), brute force on a tiny input,
or a published known answer.  CPU only.
"""
import math
import os

import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator
from scipy.spatial.transform import Rotation

from workloads import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def paper_constants():
    out = {}
    for line in open(os.path.join(GOLD, "paper_constants.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()[:2]
        out[k] = float(v)
    return out


# --------------------------------------------------------------------------- defaults = paper's constants
def test_default_params_are_the_papers(orc):
    c = paper_constants()
    p = orc.default_params()
    assert (p.w_long, p.w_clash, p.w_hbond) == (c["w_long"], c["w_clash"], c["w_Hbond"])
    assert p.long_dmax == c["d_max"] and p.hb_dclash == c["d_clash_hb"]
    assert (p.hb_mu, p.hb_sigma, p.hb_dmax) == (c["hb_mu"], c["hb_sigma"], c["hb_dmax"])
    assert p.w_tor == c["w_tor"] and p.lr == c["adam_lr"] and p.beta == c["beta"]
    # beta makes P(accept) = 0.5 for dE = 10
    assert abs(math.exp(-p.beta * 10.0) - c["p_accept_dE10"]) < 2e-3
    # G2: E_long is Vina's second Gaussian exp(-((d_surf - 3)/2)^2)
    assert p.long_mu == 3.0 and p.long_two_sigma2 == 4.0


# --------------------------------------------------------------------------- O2 pair function, closed forms
R_NON = (1.7, 0)      # radius, role : plain
R_DON = (1.6, 1)      # donor
R_ACC = (1.8, 2)      # acceptor


def test_pair_long_closed_forms(orc):
    p = orc.default_params()
    dvdw = R_NON[0] + R_NON[0]
    e, de = orc.pair(p, *R_NON, *R_NON, dvdw + 3.0)          # Gaussian centre: L = -1
    assert e == pytest.approx(-0.2, abs=1e-15) and de == pytest.approx(0.0, abs=1e-15)
    # Vina's second Gaussian drops to exp(-1) at surface distance 3 +/- 2
    for s in (+2.0, -2.0):
        d = dvdw + 3.0 + s
        e, _ = orc.pair(p, *R_NON, *R_NON, d)
        clash = 0.0                                           # d >= dvdw here (3.4+1 = 4.4 > 3.4)
        assert e - clash == pytest.approx(-0.2 * math.exp(-1.0), rel=1e-14)
    # cutoff: zero at and beyond d_max = 10, non-zero just inside
    assert orc.pair(p, *R_NON, *R_NON, 10.0) == (0.0, 0.0)
    assert orc.pair(p, *R_NON, *R_NON, 25.0) == (0.0, 0.0)
    assert orc.pair(p, *R_NON, *R_NON, 10.0 - 1e-9)[0] < 0.0


def test_pair_clash_closed_forms(orc):
    p = orc.default_params(w_long=0.0, w_hbond=0.0)
    dvdw = R_NON[0] + R_NON[0]
    e, de = orc.pair(p, *R_NON, *R_NON, dvdw / math.e)        # -ln(1/e) = 1 -> 10 * 1
    assert e == pytest.approx(10.0, rel=1e-14)
    assert de == pytest.approx(-10.0 / (dvdw / math.e), rel=1e-14)
    assert orc.pair(p, *R_NON, *R_NON, dvdw)[0] == 0.0         # indicator is strict
    assert orc.pair(p, *R_NON, *R_NON, dvdw * (1 - 1e-12))[0] == pytest.approx(0.0, abs=1e-10)  # continuous
    # H-bond pair: d_clash = 2.6; reading G3 -> no penalty for 2.6 <= d < d_vdw
    assert orc.pair(p, *R_DON, *R_ACC, 2.6 + 1e-9)[0] == 0.0
    assert orc.pair(p, *R_DON, *R_ACC, 3.0)[0] == 0.0
    assert orc.pair(p, *R_DON, *R_ACC, 2.6 / math.e)[0] == pytest.approx(10.0, rel=1e-14)
    # paper-literal indicator [d < d_vdw] (kept as an oracle-only switch): negative "penalty" in (2.6, d_vdw)
    pl = orc.default_params(w_long=0.0, w_hbond=0.0, clash_literal=1)
    assert orc.pair(pl, *R_DON, *R_ACC, 3.0)[0] == pytest.approx(-10.0 * math.log(3.0 / 2.6), rel=1e-14)
    # two donors are not an H-bond pair: d_clash = d_vdw
    assert orc.pair(p, *R_DON, *R_DON, 3.0)[0] == pytest.approx(-10.0 * math.log(3.0 / 3.2), rel=1e-14)
    # floor (G4): finite at d -> 0, derivative zero below the floor
    e0, de0 = orc.pair(p, *R_NON, *R_NON, 0.0)
    assert e0 == pytest.approx(10.0 * math.log(dvdw / 0.05), rel=1e-14) and de0 == 0.0


def test_pair_hbond_closed_forms(orc):
    p = orc.default_params(w_long=0.0, w_clash=0.0)
    assert orc.pair(p, *R_DON, *R_ACC, 2.88)[0] == pytest.approx(-0.6, rel=1e-15)          # Gaussian centre
    assert orc.pair(p, *R_ACC, *R_DON, 2.88)[0] == pytest.approx(-0.6, rel=1e-15)          # symmetric in roles
    assert orc.pair(p, *R_DON, *R_ACC, 3.4 - 1e-12)[0] == pytest.approx(-0.6 * 0.22263, rel=5e-5)  # SURVEY section 4 (5 digits)
    assert orc.pair(p, *R_DON, *R_ACC, 3.4)[0] == 0.0
    assert orc.pair(p, *R_DON, *R_DON, 2.88)[0] == 0.0                                     # donor/donor: none
    assert orc.pair(p, *R_NON, *R_ACC, 2.88)[0] == 0.0
    both = (1.7, 3)
    assert orc.pair(p, *both, *both, 2.88)[0] == pytest.approx(-0.6, rel=1e-15)           # role 3 = donor+acceptor


def test_pair_total_is_weighted_sum(orc):
    """Eq.E_dock: the three terms add linearly with their weights."""
    d = 2.4
    full = orc.pair(orc.default_params(), *R_DON, *R_ACC, d)
    parts = [orc.pair(orc.default_params(**{k: 0.0 for k in ks}), *R_DON, *R_ACC, d)
             for ks in (("w_clash", "w_hbond"), ("w_long", "w_hbond"), ("w_long", "w_clash"))]
    assert full[0] == pytest.approx(sum(x[0] for x in parts), rel=1e-14)
    assert full[1] == pytest.approx(sum(x[1] for x in parts), rel=1e-14)


def test_pair_derivative_vs_central_difference(orc):
    p = orc.default_params()
    rng = np.random.default_rng(0)
    edges = [10.0, 3.4, 2.6, 0.05]
    for a, b in ((R_NON, R_NON), (R_DON, R_ACC), (R_NON, R_ACC), ((2.25, 3), (1.5, 3))):
        ed = edges + [a[0] + b[0]]
        for d in rng.uniform(0.2, 11.0, size=200):
            if min(abs(d - x) for x in ed) < 1e-3:
                continue
            h = 1e-6
            fd = (orc.pair(p, *a, *b, d + h)[0] - orc.pair(p, *a, *b, d - h)[0]) / (2 * h)
            assert orc.pair(p, *a, *b, d)[1] == pytest.approx(fd, rel=1e-6, abs=1e-7)


# --------------------------------------------------------------------------- O3/O4 brute force <-> grid
@pytest.fixture(scope="module")
def small_system(orc):
    rng = np.random.default_rng(7)
    radius, role = synth.type_table(8)
    ty = orc.Types(radius, role)
    rec_xyz = rng.uniform(0, 6.0, size=(40, 3))
    rec_type = rng.integers(0, 8, size=40)
    p = orc.default_params()
    G = orc.build_grid(p, ty, rec_xyz, rec_type, (0.5, 0.25, 0.0), (9, 8, 7), 0.375)
    return dict(p=p, ty=ty, rec_xyz=rec_xyz, rec_type=rec_type, G=G, radius=radius, role=role)


def test_field_of_one_atom_is_the_pair_function(orc):
    radius, role = synth.type_table(8)
    ty = orc.Types(radius, role)
    p = orc.default_params()
    for s, t, d in ((0, 1, 3.3), (2, 3, 2.9), (6, 6, 2.0), (5, 7, 7.7)):
        f = orc.field_brute(p, ty, [[1.0, 2.0, 3.0]], [s], t, [1.0, 2.0 + d, 3.0])
        assert f == pytest.approx(orc.pair(p, radius[s], role[s], radius[t], role[t], d)[0], rel=1e-13)


def test_field_is_additive_over_receptor_atoms(orc, small_system):
    S = small_system
    x = [2.2, 3.1, 1.7]
    tot = orc.field_brute(S["p"], S["ty"], S["rec_xyz"], S["rec_type"], 3, x)
    parts = sum(orc.field_brute(S["p"], S["ty"], S["rec_xyz"][i:i + 1], S["rec_type"][i:i + 1], 3, x)
                for i in range(40))
    assert tot == pytest.approx(parts, rel=1e-12)


def test_grid_equals_brute_force_at_every_node(orc, small_system):
    S = small_system
    G = S["G"]
    nt, nz, ny, nx = G.g.shape
    assert (nt, nz, ny, nx) == (8, 7, 8, 9)
    rng = np.random.default_rng(1)
    for _ in range(300):
        t, k, j, i = rng.integers(nt), rng.integers(nz), rng.integers(ny), rng.integers(nx)
        x = G.origin + G.spacing * np.array([i, j, k])
        f = orc.field_brute(S["p"], S["ty"], S["rec_xyz"], S["rec_type"], int(t), x)
        assert G.g[t, k, j, i] == np.float32(f)              # x fastest, rounded once to fp32


# --------------------------------------------------------------------------- O5 trilinear interpolation
def test_trilinear_exact_on_nodes(orc, small_system):
    S = small_system
    G = S["G"]
    nt, nz, ny, nx = G.g.shape
    for t in range(nt):
        for (i, j, k) in ((0, 0, 0), (nx - 1, ny - 1, nz - 1), (3, 4, 5), (nx - 1, 0, 2), (1, ny - 1, 0)):
            x = G.origin + G.spacing * np.array([i, j, k])
            e, _ = orc.interp(S["p"], G, t, x)
            assert e == pytest.approx(float(G.g[t, k, j, i]), rel=1e-13, abs=1e-13)


def test_trilinear_exact_on_trilinear_fields(orc):
    """A field a + b x + c y + d z + e xy + f yz + g xz + h xyz is reproduced exactly, gradient analytic."""
    rng = np.random.default_rng(3)
    co = rng.normal(size=8)
    origin, h, n = np.array([-1.0, 2.0, 0.5]), 0.5, (6, 5, 7)         # nx, ny, nz ; h exact in binary
    X, Y, Z = np.meshgrid(*(origin[c] + h * np.arange(n[c]) for c in range(3)), indexing="ij")

    def F(x, y, z):
        return co[0] + co[1] * x + co[2] * y + co[3] * z + co[4] * x * y + co[5] * y * z + co[6] * x * z + co[7] * x * y * z

    vals = F(X, Y, Z).transpose(2, 1, 0)[None]                          # [1][z][y][x]
    G = orc.Grid(vals.astype(np.float32), origin, h)
    g64 = G.g.astype(np.float64)[0].transpose(2, 1, 0)                  # what the oracle sees (fp32-rounded nodes)
    rgi = RegularGridInterpolator(tuple(origin[c] + h * np.arange(n[c]) for c in range(3)), g64, method="linear")
    p = orc.default_params()
    for _ in range(200):
        x = origin + rng.uniform(0.0, 1.0, size=3) * h * (np.array(n) - 1)
        e, g = orc.interp(p, G, 0, x)
        assert e == pytest.approx(F(*x), rel=2e-6, abs=2e-6)            # fp32 node rounding only
        assert e == pytest.approx(float(rgi(x)[0]), rel=1e-12, abs=1e-12)   # library pin
        ga = np.array([co[1] + co[4] * x[1] + co[6] * x[2] + co[7] * x[1] * x[2],
                       co[2] + co[4] * x[0] + co[5] * x[2] + co[7] * x[0] * x[2],
                       co[3] + co[5] * x[1] + co[6] * x[0] + co[7] * x[0] * x[1]])
        assert g == pytest.approx(ga, rel=1e-4, abs=1e-4)


def test_trilinear_matches_scipy_and_fd_on_a_real_grid(orc, small_system):
    S = small_system
    G = S["G"]
    nt, nz, ny, nx = G.g.shape
    axes = tuple(G.origin[c] + G.spacing * np.arange(m) for c, m in enumerate((nx, ny, nz)))
    rng = np.random.default_rng(5)
    for t in (0, 2, 6):
        rgi = RegularGridInterpolator(axes, G.g[t].astype(np.float64).transpose(2, 1, 0), method="linear")
        for _ in range(100):
            cell = np.array([rng.integers(nx - 1), rng.integers(ny - 1), rng.integers(nz - 1)])
            frac = rng.uniform(0.05, 0.95, size=3)                      # strictly inside a cell
            x = G.origin + G.spacing * (cell + frac)
            e, g = orc.interp(S["p"], G, t, x)
            assert e == pytest.approx(float(rgi(x)[0]), rel=1e-12, abs=1e-12)
            h = 1e-6
            for c in range(3):
                dx = np.zeros(3); dx[c] = h
                fd = (orc.interp(S["p"], G, t, x + dx)[0] - orc.interp(S["p"], G, t, x - dx)[0]) / (2 * h)
                assert g[c] == pytest.approx(fd, rel=1e-6, abs=1e-6 * max(1.0, abs(e)))


def test_wall_outside_the_grid(orc, small_system):
    """G8: clamp + quadratic wall k (x - x_clamped)^2; the interpolant's own gradient is zeroed on a clamped axis."""
    S = small_system
    G = S["G"]
    nt, nz, ny, nx = G.g.shape
    hi = G.origin + G.spacing * (np.array([nx, ny, nz]) - 1)
    x_in = G.origin + G.spacing * np.array([2.3, 3.6, 1.2])
    for axis, sign, dist in ((0, +1, 0.7), (1, -1, 1.3), (2, +1, 0.01)):
        x = x_in.copy()
        edge = hi[axis] if sign > 0 else G.origin[axis]
        x[axis] = edge + sign * dist
        xc = x.copy(); xc[axis] = edge
        e, g = orc.interp(S["p"], G, 1, x)
        ec, gc = orc.interp(S["p"], G, 1, xc)
        assert e == pytest.approx(ec + 10.0 * dist ** 2, rel=1e-12)
        assert g[axis] == pytest.approx(sign * 2 * 10.0 * dist, rel=1e-12)
        other = [c for c in range(3) if c != axis]
        assert g[other] == pytest.approx(gc[other], rel=1e-12)


# --------------------------------------------------------------------------- O8 forward kinematics
def hand_ligand(orc):
    """Butane-like chain along z with one torsion about the z axis, plus an off-axis tail."""
    ref = np.array([[1.0, 0.0, -1.0], [0.0, 0.0, 0.0], [0.0, 0.0, 1.5], [1.2, 0.3, 2.0], [1.5, -0.7, 3.0]])
    return orc.Ligand(ref, [0, 1, 2, 3, 4], [0, 0, 1, 1, 1], tor_a=[1], tor_b=[2], tor_parent=[-1],
                      pairs=np.zeros((0, 2), np.uint8))


def test_fk_identity_reproduces_reference(orc):
    L = hand_ligand(orc)
    assert orc.fk(L, [0, 0, 0, 1, 0, 0, 0, 0.0]) == pytest.approx(L.ref, abs=1e-15)


def test_fk_one_torsion_about_z_is_the_textbook_matrix(orc):
    L = hand_ligand(orc)
    th = 0.7
    x = orc.fk(L, [0, 0, 0, 1, 0, 0, 0, th])
    Rz = np.array([[math.cos(th), -math.sin(th), 0], [math.sin(th), math.cos(th), 0], [0, 0, 1]])
    assert x[:3] == pytest.approx(L.ref[:3], abs=1e-15)                 # root side + axis atoms fixed
    assert x[3:] == pytest.approx((Rz @ L.ref[3:].T).T, abs=1e-14)      # right-handed about a -> b = +z


def test_fk_rigid_part_matches_scipy_rotation(orc):
    rng = np.random.default_rng(11)
    batch = synth.ligands([20], [0], 8, seed=5)
    L = orc.ligand_from_batch(batch, 0)
    assert L.T == 0
    for _ in range(20):
        q = rng.normal(size=4); q /= np.linalg.norm(q)
        t = rng.normal(size=3) * 5
        x = orc.fk(L, np.concatenate([t, q]))
        R = Rotation.from_quat([q[1], q[2], q[3], q[0]])                # scipy is scalar-last
        assert x == pytest.approx(R.apply(L.ref) + t, abs=1e-13)
        assert orc.fk(L, np.concatenate([t, -q])) == pytest.approx(x, abs=1e-13)       # q and -q
        assert orc.fk(L, np.concatenate([t, 3.7 * q])) == pytest.approx(x, abs=1e-13)  # input renormalised


def _dihedral(p0, p1, p2, p3):
    b1, b2, b3 = p1 - p0, p2 - p1, p3 - p2
    n1, n2 = np.cross(b1, b2), np.cross(b2, b3)
    return math.atan2(np.dot(np.cross(n1, n2), b2 / np.linalg.norm(b2)), np.dot(n1, n2))


def test_fk_preserves_internal_coordinates_and_drives_dihedrals(orc):
    rng = np.random.default_rng(13)
    batch = synth.ligands([30, 24, 40], [6, 3, 9], 16, seed=9)
    for li in range(3):
        L = orc.ligand_from_batch(batch, li)
        bonds = batch.one(li)["bond_ab"].astype(int)
        nbr = {a: set() for a in range(L.n)}
        for a, b in bonds:
            nbr[a].add(b); nbr[b].add(a)
        rot = {(int(a), int(b)) for a, b in zip(L.tor_a, L.tor_b)}
        is_rot = lambda a, b: (a, b) in rot or (b, a) in rot
        for _ in range(5):
            pose = np.concatenate([rng.normal(size=3) * 4, rng.normal(size=4), rng.uniform(-np.pi, np.pi, L.T)])
            x = orc.fk(L, pose)
            pose2 = pose.copy(); pose2[7:] += 2 * np.pi
            assert orc.fk(L, pose2) == pytest.approx(x, abs=1e-12)       # theta and theta + 2 pi
            for a, b in bonds:                                           # bond lengths
                assert np.linalg.norm(x[a] - x[b]) == pytest.approx(np.linalg.norm(L.ref[a] - L.ref[b]), abs=1e-12)
            for b in range(L.n):                                         # bond angles
                nb = sorted(nbr[b])
                for i in range(len(nb)):
                    for j in range(i + 1, len(nb)):
                        a, c = nb[i], nb[j]
                        assert np.linalg.norm(x[a] - x[c]) == pytest.approx(np.linalg.norm(L.ref[a] - L.ref[c]), abs=1e-12)
            for b, c in bonds:                                           # dihedrals a-b-c-d
                for a in nbr[b] - {c}:
                    for d in nbr[c] - {b}:
                        phi, phi0 = _dihedral(x[a], x[b], x[c], x[d]), _dihedral(*L.ref[[a, b, c, d]])
                        delta = (phi - phi0 + np.pi) % (2 * np.pi) - np.pi
                        if not is_rot(b, c):
                            assert abs(delta) < 1e-10                    # not driven: unchanged
                        else:
                            k = [i for i in range(L.T) if {int(L.tor_a[i]), int(L.tor_b[i])} == {b, c}][0]
                            th = pose[7 + k] if (int(L.tor_a[k]), int(L.tor_b[k])) == (b, c) else pose[7 + k]
                            want = (th + np.pi) % (2 * np.pi) - np.pi
                            assert abs((delta - want + np.pi) % (2 * np.pi) - np.pi) < 1e-10   # driven by exactly theta_k


def test_derive_pairs_matches_brute_force_bfs(orc):
    """O6: pairs = {a<b : graph distance >= 4 and different fragment}; independent BFS in Python."""
    batch = synth.ligands([12, 30, 50], [2, 6, 10], 8, seed=21)
    for li in range(3):
        d = batch.one(li)
        n = len(d["atom_type"])
        nbr = {a: [] for a in range(n)}
        for a, b in d["bond_ab"].astype(int):
            nbr[a].append(b); nbr[b].append(a)
        want = []
        for a in range(n):
            dist = {a: 0}; frontier = [a]
            while frontier:
                nxt = []
                for u in frontier:
                    for v in nbr[u]:
                        if v not in dist:
                            dist[v] = dist[u] + 1; nxt.append(v)
                frontier = nxt
            for b in range(a + 1, n):
                if dist[b] >= 4 and d["atom_frag"][a] != d["atom_frag"][b]:
                    want.append((a, b))
        got = orc.derive_pairs(d["atom_frag"], d["bond_ab"])
        assert [tuple(x) for x in got.astype(int)] == want
        assert len(want) > 0


# --------------------------------------------------------------------------- O6/O7/O9 score + gradient
@pytest.fixture(scope="module")
def dock_system(orc):
    """Small receptor + grid + 3 ligands, oracle-built grid."""
    rec = synth.receptor(120, 15.0, 8, seed=31, grid_n=41, pocket_radius=4.0)
    radius, role = synth.type_table(8)
    ty = orc.Types(radius, role)
    p = orc.default_params()
    G = orc.build_grid(p, ty, rec.xyz, rec.type, rec.origin, rec.dims, rec.spacing)
    batch = synth.ligands([12, 20, 26], [2, 4, 6], 8, seed=41)
    return dict(rec=rec, ty=ty, p=p, G=G, batch=batch, L=[orc.ligand_from_batch(batch, i) for i in range(3)])


def test_intra_energy_is_rigid_invariant_and_obeys_newton(orc, dock_system):
    S = dock_system
    rng = np.random.default_rng(17)
    zero = orc.Grid(np.zeros((8, 41, 41, 41), np.float32), S["rec"].origin, S["rec"].spacing)
    for L in S["L"]:
        th = rng.uniform(-np.pi, np.pi, L.T)
        ref_e = None
        for _ in range(6):
            pose = np.concatenate([7.5 + rng.uniform(-1, 1, 3), rng.normal(size=4), th])
            e, g, x, ga = orc.score_grad(S["p"], S["ty"], zero, L, pose)
            assert e[1] == 0.0                                           # zero grid, inside the box: no inter/wall
            ref_e = e[2] if ref_e is None else ref_e
            assert e[2] == pytest.approx(ref_e, rel=1e-12, abs=1e-12)    # invariant under (t, q)
            assert ga.sum(axis=0) == pytest.approx(0.0, abs=1e-10)       # sum of internal forces = 0
            assert np.cross(x, ga).sum(axis=0) == pytest.approx(0.0, abs=1e-9)   # and of internal torques
            assert g[:6] == pytest.approx(0.0, abs=1e-9)                 # so no rigid-body gradient
        assert ref_e != 0.0


def test_inter_energy_is_sum_of_per_atom_interpolations(orc, dock_system):
    S = dock_system
    L = S["L"][1]
    pose = np.concatenate([[7.4, 7.7, 7.2], [0.3, -0.5, 0.2, 0.8], [0.5, -1.0, 2.0, 0.1]])
    e, g, x, ga = orc.score_grad(S["p"], S["ty"], S["G"], L, pose)
    tot = sum(orc.interp(S["p"], S["G"], int(L.type[a]), x[a])[0] for a in range(L.n))
    assert e[1] == pytest.approx(tot, rel=1e-13)
    assert e[0] == pytest.approx(e[1] + e[2], rel=1e-14)


def _quat_left_mul_rotvec(q_wxyz, v):
    r = Rotation.from_rotvec(v) * Rotation.from_quat([q_wxyz[1], q_wxyz[2], q_wxyz[3], q_wxyz[0]])
    x, y, z, w = r.as_quat()
    return np.array([w, x, y, z])


def _safe_pose(orc, S, L, rng, margin=1e-3):
    """A pose with no atom within `margin` (grid units) of a cell face and no pair within `margin` of an indicator edge."""
    G = S["G"]
    for _ in range(200):
        pose = np.concatenate([7.5 + rng.uniform(-2.5, 2.5, 3), rng.normal(size=4), rng.uniform(-np.pi, np.pi, L.T)])
        pose[3:7] /= np.linalg.norm(pose[3:7])
        x = orc.fk(L, pose)
        u = (x - G.origin) / G.spacing
        if np.any(u < 0.01) or np.any(u > 39.99) or np.min(np.abs(u - np.rint(u))) < margin:
            continue
        ok = True
        for a, b in L.pairs.astype(int):
            d = np.linalg.norm(x[a] - x[b])
            r = S["ty"].radius[L.type[a]] + S["ty"].radius[L.type[b]]
            if min(abs(d - e) for e in (10.0, 3.4, 2.6, r, 0.05)) < margin:
                ok = False
        if ok:
            return pose
    raise RuntimeError("no safe pose")


def test_gradient_matches_central_differences(orc, dock_system):
    S = dock_system
    rng = np.random.default_rng(23)
    h = 1e-5
    E = lambda L, pose: orc.score_grad(S["p"], S["ty"], S["G"], L, pose, want_grad=False)[0][0]
    for L in S["L"]:
        for _ in range(4):
            pose = _safe_pose(orc, S, L, rng)
            e, g, x, ga = orc.score_grad(S["p"], S["ty"], S["G"], L, pose)
            assert g[:3] == pytest.approx(ga.sum(axis=0), rel=1e-12, abs=1e-12)      # translation row = sum of forces
            scale = max(1.0, np.abs(g).max())
            for c in range(3):
                d = np.zeros_like(pose); d[c] = h
                assert g[c] == pytest.approx((E(L, pose + d) - E(L, pose - d)) / (2 * h), abs=2e-5 * scale)
            for c in range(3):                                                         # world-frame rotation about t
                v = np.zeros(3); v[c] = h
                pp, pm = pose.copy(), pose.copy()
                pp[3:7] = _quat_left_mul_rotvec(pose[3:7], v)
                pm[3:7] = _quat_left_mul_rotvec(pose[3:7], -v)
                assert g[3 + c] == pytest.approx((E(L, pp) - E(L, pm)) / (2 * h), abs=2e-5 * scale)
            for k in range(L.T):
                d = np.zeros_like(pose); d[7 + k] = h
                assert g[6 + k] == pytest.approx((E(L, pose + d) - E(L, pose - d)) / (2 * h), abs=2e-5 * scale)


# --------------------------------------------------------------------------- O10 Philox, uniforms
def test_philox_known_answers(orc):
    n = 0
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert orc.philox4x32_10(w[0:4], w[4:6]) == w[6:10]
        n += 1
    assert n == 3


def test_uniform_mapping(orc):
    """u = ((r >> 9) + 0.5) 2^-23: strictly inside (0,1), exact in fp32, counter = (chain, step, ligand, purpose)."""
    r = orc.philox4x32_10([5, 6, 7, 1], [0x89abcdef, 0x01234567])
    u = orc.uniform4(0x0123456789abcdef, 5, 6, 7, 1)
    for ri, ui in zip(r, u):
        assert ui == ((ri >> 9) + 0.5) / 2 ** 23
        assert 0.0 < ui < 1.0 and float(np.float32(ui)) == ui
    us = np.concatenate([orc.uniform4(3, c, 0, 0, 0) for c in range(5000)])
    assert abs(us.mean() - 0.5) < 0.01 and abs(us.var() - 1 / 12) < 0.005
    assert not np.array_equal(orc.uniform4(3, 1, 0, 0, 0), orc.uniform4(3, 0, 1, 0, 0))


# --------------------------------------------------------------------------- O11 init
def test_init_pose_distribution(orc, dock_system):
    L = dock_system["L"][2]
    c, R = np.array([7.5, 7.5, 7.5]), 4.0
    P = np.array([orc.init_pose(L, 0, ch, 3, c, R) for ch in range(4000)])
    r = np.linalg.norm(P[:, :3] - c, axis=1)
    assert r.max() <= R
    assert abs(np.mean((r / R) ** 3) - 0.5) < 0.02                       # uniform in the ball
    assert np.linalg.norm(P[:, 3:7], axis=1) == pytest.approx(1.0, abs=1e-12)
    assert np.abs(P[:, 3:7].mean(axis=0)).max() < 0.03                   # uniform on S^3: zero mean ...
    assert np.mean(P[:, 3:7] ** 2, axis=0) == pytest.approx(0.25, abs=0.01)  # ... and isotropic
    assert np.all(P[:, 7:] >= -np.pi) and np.all(P[:, 7:] < np.pi)
    assert np.abs(P[:, 7:].mean(axis=0)).max() < 0.12
    assert np.array_equal(P[5], orc.init_pose(L, 0, 5, 3, c, R))         # counter-based: reproducible


# --------------------------------------------------------------------------- O12 Adam + Metropolis
def one_atom_system(orc):
    """One atom outside a zero grid on +x: E = k_wall (x - x_max)^2, a 1-D quadratic in the translation."""
    L = orc.Ligand(np.zeros((1, 3)), [0], [0], [], [], [], pairs=np.zeros((0, 2), np.uint8))
    G = orc.Grid(np.zeros((1, 4, 4, 4), np.float32), (0, 0, 0), 1.0)     # x_max = 3
    ty = orc.Types([1.7], [0])
    return L, G, ty


def test_adam_first_step_and_torch_reference(orc):
    import torch
    L, G, ty = one_atom_system(orc)
    box = ([-100.0] * 3, [100.0] * 3)
    x0 = 5.0
    pose0 = [x0, 1.5, 1.5, 1, 0, 0, 0]
    for n_refine in (1, 2, 5):
        p = orc.default_params(pert_trans=0.0, pert_rot=0.0, n_refine=n_refine)
        e0 = orc.score_grad(p, ty, G, L, pose0)[0][0]
        assert e0 == pytest.approx(10.0 * (x0 - 3.0) ** 2, rel=1e-14)
        pose, ec, rec = orc.mc_step(p, ty, G, L, 0, 0, 0, 0, *box, pose0, e0)
        assert rec.accept == 1                                           # downhill: always accepted (G15)
        xt = torch.tensor([x0], dtype=torch.float64, requires_grad=True)
        opt = torch.optim.Adam([xt], lr=0.1)                             # PyTorch defaults = G12
        for _ in range(n_refine):
            opt.zero_grad()
            (10.0 * (xt - 3.0) ** 2).sum().backward()
            opt.step()
        assert pose[0] == pytest.approx(float(xt.detach()[0]), rel=1e-12)
        assert pose[1:3] == pytest.approx([1.5, 1.5], abs=0)             # zero gradient -> zero Adam step
        assert ec == pytest.approx(10.0 * (pose[0] - 3.0) ** 2, rel=1e-13)
        if n_refine == 1:                                                # hand value: -lr g / (|g| + eps)
            g = 2 * 10.0 * (x0 - 3.0)
            assert pose[0] == pytest.approx(x0 - 0.1 * g / (abs(g) + 1e-8), rel=1e-15)


def test_metropolis_acceptance_probability(orc):
    """P(accept | dE = +10) = exp(-0.69) = 0.5016; dE <= 0 always accepts; large beta never goes uphill."""
    L, G, ty = one_atom_system(orc)
    box = ([-100.0] * 3, [100.0] * 3)
    pose0 = [5.0, 1.5, 1.5, 1, 0, 0, 0]
    p = orc.default_params(pert_trans=0.0, pert_rot=0.0, lr=0.0)         # proposal == current pose
    e_here = orc.score_grad(p, ty, G, L, pose0)[0][0]
    n, acc = 20000, 0
    for i in range(n):
        _, _, rec = orc.mc_step(p, ty, G, L, 1, i % 100, i // 100, 2, *box, pose0, e_here - 10.0)
        assert rec.e_prop - rec.e_cur == pytest.approx(10.0, rel=1e-12)
        assert rec.accept == int(rec.u < math.exp(-0.69))
        acc += rec.accept
    assert abs(acc / n - 0.5016) < 4 * math.sqrt(0.25 / n)
    for i in range(200):
        _, _, rec = orc.mc_step(p, ty, G, L, 1, i, 0, 0, *box, pose0, e_here)          # dE = 0
        assert rec.accept == 1
        _, _, rec = orc.mc_step(p, ty, G, L, 1, i, 0, 0, *box, pose0, e_here + 3.0)    # dE < 0
        assert rec.accept == 1
    pb = orc.default_params(pert_trans=0.0, pert_rot=0.0, lr=0.0, beta=1e3)
    for i in range(200):
        _, _, rec = orc.mc_step(pb, ty, G, L, 1, i, 0, 0, *box, pose0, e_here - 1.0)
        assert rec.accept == 0


def test_perturbation_entities_and_ranges(orc, dock_system):
    """G11: entity uniform over {translation, rotation, each torsion}; translation stays in the box."""
    S = dock_system
    L = S["L"][1]                                                        # T = 4 -> 6 entities
    p = orc.default_params(lr=0.0)                                       # isolate the perturbation
    rec_ = S["rec"]
    pose0 = np.concatenate([rec_.pocket_center, [1, 0, 0, 0], [0.1, 0.2, 0.3, 0.4]])
    counts = np.zeros(L.T + 2, int)
    for i in range(3000):
        pose, ec, rec = orc.mc_step(p, S["ty"], S["G"], L, 9, i, 0, 0, rec_.box_min, rec_.box_max, pose0, 1e9)
        assert rec.accept == 1                                           # e_cur huge -> always accepted
        counts[rec.entity] += 1
        changed_t = not np.array_equal(pose[:3], pose0[:3])
        changed_q = not np.allclose(pose[3:7], pose0[3:7], atol=1e-15)
        changed_th = [k for k in range(L.T) if abs(pose[7 + k] - pose0[7 + k]) > 1e-9]   # wrap() rounds in the last bit
        assert (changed_t, changed_q, changed_th) == (rec.entity == 0, rec.entity == 1,
                                                      [rec.entity - 2] if rec.entity >= 2 else [])
        assert np.all(pose[:3] >= rec_.box_min) and np.all(pose[:3] <= rec_.box_max)
        assert np.all(np.abs(pose[:3] - pose0[:3]) <= 2.0)
        assert abs(np.linalg.norm(pose[3:7]) - 1) < 1e-12
        if rec.entity == 1:
            ang = 2 * math.acos(min(1.0, abs(pose[3])))
            assert ang <= 0.5 * math.sqrt(3) + 1e-12
    assert counts.min() > 3000 / 6 * 0.8


# --------------------------------------------------------------------------- O12: rotation / torsion branch of the MC step
def _rigid_entity_counter(orc, L, seed, lig, want):
    """(chain, step) whose perturbation block picks entity `want` (0 translation, 1 rotation, 2+k torsion k)."""
    for chain in range(64):
        for step in range(64):
            if int(math.floor(orc.uniform4(seed, chain, step, lig, 0)[0] * (L.T + 2))) == want:
                return chain, step
    raise RuntimeError("no counter found")


def _rot(q_wxyz):
    return Rotation.from_quat([q_wxyz[1], q_wxyz[2], q_wxyz[3], q_wxyz[0]])


def test_adam_step_is_first_order_descent_on_all_components(orc, dock_system):
    """O12 / G9 / G14.  With zero perturbation amplitudes the proposal is the current pose; the first Adam step is
    delta_i = -lr g_i / (|g_i| + eps) = -lr sign(g_i) on every one of the 6+T tangent components (translation, WORLD-frame
    rotation vector about t, torsions).  Two pins that do not retype the update:
      (a) the descent identity  E(pose') - E(pose) = sum_i g_i delta_i + O(lr^2) = -lr sum_i |g_i|, with g the gradient
          that test_gradient_matches_central_differences pins against finite differences -- it fails for a body-frame
          composition q (x) exp(d), a quarter angle in exp_q, a sign or an index slip in the torsion update;
      (b) the returned pose equals t - lr sign(g_t), Rotation.from_rotvec(-lr sign(g_w)) * Rotation(q) (scipy composes),
          theta - lr sign(g_theta)."""
    S = dock_system
    rng = np.random.default_rng(101)
    lr = 1e-5
    p = orc.default_params(pert_trans=0.0, pert_rot=0.0, lr=lr, n_refine=1)
    rec_ = S["rec"]
    E = lambda L, pose: orc.score_grad(p, S["ty"], S["G"], L, pose, want_grad=False)[0][0]
    n_sign_mixed = 0
    for li, L in enumerate(S["L"]):
        for trial in range(6):
            pose0 = _safe_pose(orc, S, L, rng, margin=5e-3)
            pose0[:3] = np.clip(pose0[:3], rec_.box_min + 0.01, rec_.box_max - 0.01)
            x = orc.fk(L, pose0)
            u = (x - S["G"].origin) / S["G"].spacing
            if np.min(np.abs(u - np.rint(u))) < 5e-3:
                continue
            e0, g, _, _ = orc.score_grad(p, S["ty"], S["G"], L, pose0)
            if np.min(np.abs(g)) < 1e-3:                      # sign(g_i) must be unambiguous
                continue
            chain, step = _rigid_entity_counter(orc, L, 5, li, trial % 2)        # entity 0 or 1: amplitudes are zero
            pose1, e1, rec = orc.mc_step(p, S["ty"], S["G"], L, 5, chain, step, li, rec_.box_min, rec_.box_max, pose0, 1e9)
            assert rec.accept == 1 and rec.entity == trial % 2
            assert e1 == pytest.approx(E(L, pose1), rel=1e-13)
            # (a) first-order descent identity over all 6+T components
            assert e1 - e0[0] == pytest.approx(-lr * np.abs(g).sum(), rel=2e-3)
            # (b) the pose itself
            sg = g / (np.abs(g) + 1e-8)                        # Adam's first step in closed form: -lr g / (|g| + eps)
            assert pose1[:3] == pytest.approx(pose0[:3] - lr * sg[:3], abs=1e-12)
            r_exp = Rotation.from_rotvec(-lr * sg[3:6]) * _rot(pose0[3:7])
            r_got = _rot(pose1[3:7])
            assert (r_got * r_exp.inv()).magnitude() < 1e-10
            assert (r_got * (_rot(pose0[3:7]) * Rotation.from_rotvec(-lr * sg[3:6])).inv()).magnitude() > 1e-7 or \
                np.allclose(sg[3:6], 0)                        # and it is NOT the body-frame composition
            assert abs(np.linalg.norm(pose1[3:7]) - 1) < 1e-14
            assert pose1[7:] == pytest.approx(pose0[7:] - lr * sg[6:], abs=1e-12)
            n_sign_mixed += int(len(set(np.sign(g[6:]))) > 1) if L.T > 1 else 0
    assert n_sign_mixed >= 3                                   # an index swap among torsions would have shown


def test_perturbation_values_and_rotation_composition(orc, dock_system):
    """O12 / G11: with lr = 0 the accepted pose IS the perturbed pose.  Translation: t + 2 A (2u-1) per axis, clamped;
    rotation: left-multiplied (world-frame) rotation vector w = 0.5 rad (2u-1): every atom moves by
    x' - t = Rot(w)(x - t) with scipy's Rotation; torsion k: theta_k = pi (2u_1 - 1).  The uniforms are the Philox block
    (chain, step, ligand, purpose 0), pinned by the known answers."""
    S = dock_system
    rec_ = S["rec"]
    p = orc.default_params(lr=0.0)
    rng = np.random.default_rng(77)
    seen = set()
    for li, L in enumerate(S["L"]):
        pose0 = np.concatenate([rec_.pocket_center + rng.uniform(-1, 1, 3), rng.normal(size=4), rng.uniform(-3, 3, L.T)])
        pose0[3:7] /= np.linalg.norm(pose0[3:7])
        x0 = orc.fk(L, pose0)
        for i in range(60):
            chain, step = i % 7, i // 7
            u = orc.uniform4(11, chain, step, li, 0)
            pose1, _, rec = orc.mc_step(p, S["ty"], S["G"], L, 11, chain, step, li, rec_.box_min, rec_.box_max, pose0, 1e9)
            ent = int(math.floor(u[0] * (L.T + 2)))
            assert rec.entity == ent and rec.accept == 1
            seen.add(min(ent, 2))
            x1 = orc.fk(L, pose1)
            if ent == 0:
                assert pose1[:3] == pytest.approx(np.clip(pose0[:3] + 2.0 * (2 * u[1:4] - 1), rec_.box_min, rec_.box_max), abs=1e-13)
                assert x1 - pose1[:3] == pytest.approx(x0 - pose0[:3], abs=1e-12)
            elif ent == 1:
                w = 0.5 * (2 * u[1:4] - 1)
                assert x1 - pose0[:3] == pytest.approx(Rotation.from_rotvec(w).apply(x0 - pose0[:3]), abs=1e-11)
                body = (_rot(pose0[3:7]) * Rotation.from_rotvec(w)).apply(L.ref)      # the wrong (body-frame) order differs
                assert L.T > 0 or np.abs(body + pose0[:3] - x1).max() > 1e-3
            else:
                exp = pose0.copy(); exp[7 + ent - 2] = math.pi * (2 * u[1] - 1)
                assert pose1 == pytest.approx(exp, abs=1e-13)
    assert seen == {0, 1, 2}


def test_torsion_wrap_and_box_clamp_in_the_adam_update(orc, dock_system):
    """G14: torsions are wrapped into [-pi, pi) (same coordinates as the unwrapped angle), translations clamped to the box."""
    S = dock_system
    rec_ = S["rec"]
    lr = 0.1
    p = orc.default_params(pert_trans=0.0, pert_rot=0.0, lr=lr, n_refine=1)
    rng = np.random.default_rng(5)
    wrapped_up = wrapped_dn = 0
    for li, L in enumerate(S["L"]):
        for trial in range(40):
            pose0 = np.concatenate([rec_.pocket_center + rng.uniform(-1, 1, 3), rng.normal(size=4),
                                    rng.choice([-1.0, 1.0], L.T) * (math.pi - 0.05 * rng.uniform(0.1, 1.0, L.T))])
            pose0[3:7] /= np.linalg.norm(pose0[3:7])
            _, g, _, _ = orc.score_grad(p, S["ty"], S["G"], L, pose0)
            if np.min(np.abs(g)) < 1e-6:
                continue
            chain, step = _rigid_entity_counter(orc, L, 3, li, 0)
            pose1, _, rec = orc.mc_step(p, S["ty"], S["G"], L, 3, chain, step, li, rec_.box_min - 50, rec_.box_max + 50, pose0, 1e9)
            raw = pose0[7:] - lr * g[6:] / (np.abs(g[6:]) + 1e-8)         # first Adam step (pinned above)
            assert np.all(pose1[7:] >= -math.pi) and np.all(pose1[7:] < math.pi)
            k_wrap = np.rint((raw - pose1[7:]) / (2 * math.pi))
            assert pose1[7:] == pytest.approx(raw - 2 * math.pi * k_wrap, abs=1e-12)
            wrapped_up += int(np.sum(k_wrap > 0)); wrapped_dn += int(np.sum(k_wrap < 0))
            unwrapped = pose1.copy(); unwrapped[7:] = raw
            assert orc.fk(L, pose1) == pytest.approx(orc.fk(L, unwrapped), abs=1e-9)
    assert wrapped_up > 5 and wrapped_dn > 5
    # exactly -pi stays, +pi maps to -pi: the half-open interval
    L = S["L"][0]
    p0 = orc.default_params(pert_trans=0.0, pert_rot=0.0, lr=0.0)
    chain, step = _rigid_entity_counter(orc, L, 3, 0, 0)
    for th_in, th_out in ((math.pi, -math.pi), (-math.pi, -math.pi), (math.pi - 1e-9, math.pi - 1e-9)):
        pose0 = np.concatenate([rec_.pocket_center, [1, 0, 0, 0], [th_in] * L.T])
        pose1, _, _ = orc.mc_step(p0, S["ty"], S["G"], L, 3, chain, step, 0, rec_.box_min, rec_.box_max, pose0, 1e9)
        assert pose1[7:] == pytest.approx([th_out] * L.T, abs=1e-15)    # (wrap's a + pi rounds in the last bit)
    # box clamp, closed form: one atom left of a zero grid, E = k_wall x^2, g = 2 k_wall x < 0 -> step +lr, cut at box_max
    L1, G1, ty1 = one_atom_system(orc)
    pose0 = [-1.0, 1.5, 1.5, 1, 0, 0, 0]
    e0 = orc.score_grad(p, ty1, G1, L1, pose0)[0][0]
    assert e0 == pytest.approx(10.0, rel=1e-14)
    pose1, e1, rec = orc.mc_step(p, ty1, G1, L1, 0, 0, 0, 0, [-100.0] * 3, [-0.95, 100.0, 100.0], pose0, e0)
    assert pose1[0] == -0.95 and e1 == pytest.approx(10.0 * 0.95 ** 2, rel=1e-14) and rec.accept == 1
    pose1, e1, rec = orc.mc_step(p, ty1, G1, L1, 0, 0, 0, 0, [-100.0] * 3, [100.0] * 3, pose0, e0)
    assert pose1[0] == pytest.approx(-1.0 + 0.1 * 20.0 / (20.0 + 1e-8), rel=1e-14)   # unclamped: the full Adam step


# --------------------------------------------------------------------------- whole chain sanity, O13, E_screen
def test_dock_sanity_and_topk(orc, dock_system):
    S = dock_system
    rec_, L = S["rec"], S["L"][0]
    args = (S["p"], S["ty"], S["G"], L, 0, 0)
    kw = dict(box_min=rec_.box_min, box_max=rec_.box_max, centre=rec_.pocket_center, radius=rec_.pocket_radius)
    r0 = orc.dock(*args, 16, 0, **kw)
    r20 = orc.dock(*args, 16, 20, **kw, want_trace=True)
    r40 = orc.dock(*args, 16, 40, **kw)
    assert np.all(r20["e_best"] <= r0["e_best"]) and np.all(r40["e_best"] <= r20["e_best"])   # best never rises
    assert np.all(r20["e_best"] <= r20["e_cur"])
    assert r20["e_best"].min() < r0["e_best"].min()
    for c in range(16):                                                  # stored best pose scores to the stored energy
        e = orc.score_grad(S["p"], S["ty"], S["G"], L, r20["pose_best"][c], want_grad=False)[0][0]
        assert e == pytest.approx(r20["e_best"][c], rel=1e-12)
    tr = r20["trace"]
    assert np.array_equal(tr["accept"], (tr["u"] < np.exp(-0.069 * (tr["e_prop"] - tr["e_cur"]))).astype(int))
    # resumability: 20 + 20 steps (first_step = 20, from the saved state) == 40 steps
    r2 = orc.dock(*args, 16, 20, **kw, init_poses=r20["pose_cur"], first_step=20)
    assert np.minimum(r2["e_best"], r20["e_best"]) == pytest.approx(r40["e_best"], rel=1e-12)
    # O13 vs brute force
    e = np.array([3.0, -1.0, 2.0, -1.0, 5.0, -7.0])
    assert list(orc.topk(e, 4)) == [5, 1, 3, 2]                          # ties -> lower chain id
    assert list(orc.topk(r20["e_best"], 3)) == sorted(range(16), key=lambda c: (r20["e_best"][c], c))[:3]
    # Eq.E_screen
    assert orc.e_screen(-50.0, 6) == pytest.approx(-50.0 / 1.06)
    assert orc.e_screen(-50.0, 0) == -50.0


# --------------------------------------------------------------------------- O14: duplicate-removing top-k (G20)
def test_topk_cluster_constructed_cases_and_invariants(orc, dock_system):
    S = dock_system
    L = S["L"][1]
    W = 7 + L.T
    rng = np.random.default_rng(11)
    base = np.zeros(W)
    base[3] = 1.0
    base[7:] = rng.uniform(-1, 1, L.T)
    # a rigid translation by v moves every atom by v: RMSD = |v| exactly (closed form)
    shifts = np.array([0.0, 0.3, 0.9, 1.1, 2.5, 2.6, 4.0])
    poses = np.tile(base, (len(shifts), 1))
    poses[:, 0] = shifts
    x0 = orc.fk(L, poses[0])
    for i, sh in enumerate(shifts):
        xi = orc.fk(L, poses[i])
        assert np.sqrt(np.mean(np.sum((xi - x0) ** 2, axis=1))) == pytest.approx(sh, abs=1e-12)
    e = np.array([-9.0, -8.0, -7.0, -6.0, -5.0, -4.0, -3.0])
    kept, margin = orc.topk_cluster(e, poses, L, 4, 1.0)
    # 0 kept; 0.3, 0.9 are within 1 A of it; 1.1 kept; 2.5 is 1.4 from 1.1 -> kept; 2.6 within 0.1 of 2.5; 4.0 kept
    assert list(kept) == [0, 3, 4, 6] and margin == pytest.approx(0.1, abs=1e-9)
    # no threshold -> plain O13; a huge threshold -> one cluster; k larger than the number of clusters -> fewer ids
    assert list(orc.topk_cluster(e, poses, L, 4, 0.0)[0]) == list(orc.topk(e, 4))
    assert list(orc.topk_cluster(e, poses, L, 4, 100.0)[0]) == [0]
    assert list(orc.topk_cluster(e, poses, L, 7, 1.0)[0]) == [0, 3, 4, 6]
    # the energy order decides who represents a cluster: reverse the energies
    assert list(orc.topk_cluster(-e, poses, L, 3, 1.0)[0]) == [6, 5, 3]
    # invariants on random poses: kept poses are pairwise >= thr apart, every skipped better-ranked chain is a duplicate
    n_ch = 40
    P = np.zeros((n_ch, W))
    P[:, 0:3] = rng.normal(0, 0.8, (n_ch, 3))
    q = rng.normal(size=(n_ch, 4)) * 0.15 + np.array([1, 0, 0, 0])
    P[:, 3:7] = q / np.linalg.norm(q, axis=1, keepdims=True)
    P[:, 7:] = base[7:] + rng.normal(0, 0.2, (n_ch, L.T))
    E = rng.normal(size=n_ch)
    thr = 1.5
    kept, _ = orc.topk_cluster(E, P, L, 5, thr)
    X = [orc.fk(L, P[c]) for c in range(n_ch)]
    rmsd = lambda a, b: np.sqrt(np.mean(np.sum((X[a] - X[b]) ** 2, axis=1)))
    assert 1 <= len(kept) <= 5
    for i in range(len(kept)):
        for j in range(i):
            assert rmsd(kept[i], kept[j]) >= thr
    order = list(orc.topk(E, n_ch))
    last = order.index(kept[-1])
    for c in order[:last]:
        if c not in kept:
            assert any(rmsd(c, kk) < thr for kk in kept if order.index(kk) < order.index(c))


# --------------------------------------------------------------------------- direct-pair receptor mode (S:8(f) NEXT-3)
def test_direct_receptor_mode_pins(orc, dock_system):
    S = dock_system
    rec_, p, ty, G = S["rec"], S["p"], S["ty"], S["G"]
    rng = np.random.default_rng(5)
    # (1) a two-atom rigid "ligand" (atoms at -0.75 / +0.75 A on x = -2 / +2 grid steps) with both atoms exactly on grid
    #     nodes: the interpolant is exact there (O4/O5), so the grid path and the direct path -- two different routes from
    #     the paper's sums -- must agree to the grid's fp32 rounding (2 bonded atoms: no intra pair)
    one = synth.ligands([2], [0], 8, seed=3)
    assert np.array_equal(one.ref_xyz, np.array([[-0.75, 0, 0], [0.75, 0, 0]], np.float32))
    L1 = orc.ligand_from_batch(one, 0)
    for _ in range(12):
        ijk = rng.integers(4, 36, 3)
        pose = np.concatenate([rec_.origin + rec_.spacing * ijk, [1.0, 0, 0, 0]])
        eg = orc.score_grad(p, ty, G, L1, pose, want_grad=False)[0]
        ed, _, x1, _ = orc.score_grad_direct(p, ty, rec_.xyz, rec_.type, L1, pose, want_grad=False)
        assert ed[2] == 0.0 and ed[1] == pytest.approx(eg[1], rel=3e-7, abs=1e-5)
        brute = sum(orc.field_brute(p, ty, rec_.xyz, rec_.type, int(L1.type[a]), x1[a]) for a in range(2))
        assert ed[1] == pytest.approx(brute, rel=1e-13)
    # (2) same intra term as the grid path; analytic gradient vs central differences on all 6+T components
    h = 1e-5
    E = lambda L, pose: orc.score_grad_direct(p, ty, rec_.xyz, rec_.type, L, pose, want_grad=False)[0][0]
    for L in S["L"]:
        for _ in range(2):
            pose = _safe_pose(orc, S, L, rng)
            x = orc.fk(L, pose)
            dmin = np.min(np.linalg.norm(x[:, None, :] - rec_.xyz[None, :, :], axis=2))
            e, g, _, ga = orc.score_grad_direct(p, ty, rec_.xyz, rec_.type, L, pose)
            assert e[2] == orc.score_grad(p, ty, G, L, pose, want_grad=False)[0][2]
            assert g[:3] == pytest.approx(ga.sum(axis=0), rel=1e-12, abs=1e-12)
            scale = max(1.0, np.abs(g).max())
            tol = 2e-5 * scale if dmin > 0.06 else None
            if tol is None:
                continue
            for c in range(3):
                d = np.zeros_like(pose); d[c] = h
                assert g[c] == pytest.approx((E(L, pose + d) - E(L, pose - d)) / (2 * h), abs=tol)
            for c in range(3):
                v = np.zeros(3); v[c] = h
                pp, pm = pose.copy(), pose.copy()
                pp[3:7] = _quat_left_mul_rotvec(pose[3:7], v)
                pm[3:7] = _quat_left_mul_rotvec(pose[3:7], -v)
                assert g[3 + c] == pytest.approx((E(L, pp) - E(L, pm)) / (2 * h), abs=tol)
            for k in range(L.T):
                d = np.zeros_like(pose); d[7 + k] = h
                assert g[6 + k] == pytest.approx((E(L, pose + d) - E(L, pose - d)) / (2 * h), abs=tol)


# --------------------------------------------------------------------------- E_MDN (Eq.E_MDN; S:8(f) NEXT-1 groundwork)
@pytest.mark.parametrize("impl", ["python", "c"])
def test_mdn_energy_pins(impl, orc):
    """O15 under two independent transcriptions: oracle/mdn.py (plain Python) and orc_mdn_energy (C, the one orc_score_grad
    and orc_mc_step call)."""
    from scipy.stats import norm
    if impl == "python":
        from oracle import mdn
    else:
        mdn = type("M", (), {"mdn_energy": staticmethod(orc.mdn_energy)})
    rng = np.random.default_rng(3)
    one = lambda v: np.array([[[v]]], dtype=np.float64)
    # (1) one residue of one atom, one ligand atom, K = 1: E = -N(d; mu, sigma) (closed form + scipy's density)
    rec = np.zeros((1, 3)); off = np.array([0, 1])
    for d, m, s in [(3.0, 3.0, 0.5), (4.2, 3.5, 0.8), (2.0, 4.0, 1.1)]:
        E, g, dm = mdn.mdn_energy(rec, off, one(1.0), one(m), one(s), np.array([[d, 0.0, 0.0]]))
        assert dm[0, 0] == pytest.approx(d) and E == pytest.approx(-norm.pdf(d, loc=m, scale=s), rel=1e-13)
        # dE/dd = N(d) (d - mu) / sigma^2, along +x (the atom sits on the x axis, the receptor atom at the origin)
        assert g[0] == pytest.approx([norm.pdf(d, m, s) * (d - m) / s ** 2, 0, 0], rel=1e-12, abs=1e-15)
    E, _, _ = mdn.mdn_energy(rec, off, one(1.0), one(3.0), one(0.5), np.array([[3.0, 0, 0]]))
    assert E == pytest.approx(-1.0 / (0.5 * np.sqrt(2 * np.pi)), rel=1e-14)          # at d = mu: -1 / (sigma sqrt(2 pi))
    # (2) the cut-off: d_cut = 5 A, strict
    assert mdn.mdn_energy(rec, off, one(1.0), one(5.0), one(1.0), np.array([[5.0, 0, 0]]))[0] == 0.0
    assert mdn.mdn_energy(rec, off, one(1.0), one(5.0), one(1.0), np.array([[4.999, 0, 0]]))[0] < -0.39
    # (3) mixture weights: two equal components = the mean of the two single-component energies
    two = lambda a, b: np.array([[[a, b]]], dtype=np.float64)
    x = np.array([[3.3, 0, 0]])
    E2 = mdn.mdn_energy(rec, off, two(0.5, 0.5), two(3.0, 4.0), two(0.5, 0.9), x)[0]
    assert E2 == pytest.approx(0.5 * (-norm.pdf(3.3, 3.0, 0.5)) + 0.5 * (-norm.pdf(3.3, 4.0, 0.9)), rel=1e-13)
    # (4) d_ij is the MINIMUM over the residue's atoms: the nearer atom decides, the farther is irrelevant
    rec2 = np.array([[0.0, 0, 0], [0.0, 2.0, 0]]); off2 = np.array([0, 2])
    xa = np.array([[3.0, 0.0, 0.0]])
    Ea, ga, dma = mdn.mdn_energy(rec2, off2, one(1.0), one(3.2), one(0.6), xa)
    assert dma[0, 0] == pytest.approx(3.0) and Ea == pytest.approx(-norm.pdf(3.0, 3.2, 0.6), rel=1e-13)
    assert ga[0, 1] == 0.0                                                            # the gradient points along x: arg-min atom is atom 0
    # two residues add up (sum over i), two ligand atoms add up (sum over j)
    rec3 = np.array([[0.0, 0, 0], [10.0, 0, 0]]); off3 = np.array([0, 1, 2])
    x2 = np.array([[3.0, 0, 0], [7.5, 0, 0]])
    pi3 = np.ones((2, 2, 1)); mu3 = np.full((2, 2, 1), 3.0); s3 = np.full((2, 2, 1), 0.7)
    E3 = mdn.mdn_energy(rec3, off3, pi3, mu3, s3, x2)[0]
    # residue 0 sees atom 0 at 3.0 (atom 1 at 7.5: cut); residue 1 sees atom 1 at 2.5 (atom 0 at 7: cut)
    assert E3 == pytest.approx(-norm.pdf(3.0, 3.0, 0.7) - norm.pdf(2.5, 3.0, 0.7), rel=1e-13)
    # (5) analytic gradient vs central differences on a random system, away from arg-min switches and the cut-off
    rec_ = synth.receptor(120, 15.0, 8, seed=31, grid_n=41, pocket_radius=4.0)
    order, res_off = synth.residues(rec_, 8)
    rxyz = rec_.xyz[order].astype(np.float64)
    assert sorted(order) == list(range(120)) and res_off[-1] == 120 and np.all(np.diff(res_off) > 0)
    n, K = 6, 4
    pi, mu, sg = synth.gmm_params(len(res_off) - 1, n, K, seed=5)
    assert np.allclose(pi.sum(axis=2), 1.0, atol=1e-6)
    h, checked = 1e-6, 0
    for _ in range(40):
        x = rec_.pocket_center + rng.uniform(-5.0, 5.0, (n, 3))
        E, g, dm = mdn.mdn_energy(rxyz, res_off, pi, mu, sg, x)
        if np.min(np.abs(dm - 5.0)) < 1e-3:
            continue
        # skip configurations where two atoms of a residue are almost equally near (the arg-min could switch under +-h)
        near_tie = False
        for i in range(len(res_off) - 1):
            for j in range(n):
                dd = np.sort(np.linalg.norm(x[j] - rxyz[res_off[i]:res_off[i + 1]], axis=1))
                near_tie |= len(dd) > 1 and dd[1] - dd[0] < 1e-3 and dd[0] < 5.0
        if near_tie or E == 0.0:
            continue
        for j in range(n):
            for c in range(3):
                xp, xm = x.copy(), x.copy()
                xp[j, c] += h; xm[j, c] -= h
                fd = (mdn.mdn_energy(rxyz, res_off, pi, mu, sg, xp)[0] - mdn.mdn_energy(rxyz, res_off, pi, mu, sg, xm)[0]) / (2 * h)
                assert g[j, c] == pytest.approx(fd, rel=2e-6, abs=2e-8)
        checked += 1
        if checked == 3:
            break
    assert checked == 3
    # (6) invariance: a common rigid translation of receptor and ligand changes nothing
    t = np.array([1.3, -2.2, 0.7])
    E0 = mdn.mdn_energy(rxyz, res_off, pi, mu, sg, x)[0]
    assert mdn.mdn_energy(rxyz + t, res_off, pi, mu, sg, x + t)[0] == pytest.approx(E0, rel=1e-12)


def test_mdn_c_and_python_transcriptions_agree(orc):
    from oracle import mdn
    rec_ = synth.receptor(200, 18.0, 8, seed=12, grid_n=49, pocket_radius=5.0)
    order, res_off = synth.residues(rec_, 8)
    rxyz = rec_.xyz[order].astype(np.float64)
    n, K = 9, 5
    pi, mu, sg = synth.gmm_params(len(res_off) - 1, n, K, seed=2)
    rng = np.random.default_rng(8)
    for _ in range(5):
        x = rec_.pocket_center + rng.uniform(-6.0, 6.0, (n, 3))
        Ep, gp, dp = mdn.mdn_energy(rxyz, res_off, pi, mu, sg, x)
        Ec, gc, dcc = orc.mdn_energy(rxyz, res_off, pi, mu, sg, x)
        assert Ep != 0.0 and Ec == pytest.approx(Ep, rel=1e-12)
        assert np.allclose(gc, gp, rtol=1e-11, atol=1e-14) and np.allclose(dcc, dp, rtol=1e-13)


def test_total_energy_is_physics_plus_w_mdn_times_e_mdn(orc):
    """Eq.E_dock: E = 1.0 E_MDN + 0.2 E_long + 10 E_clash + 0.6 E_Hbond.  Hand case + a random system:
    orc_score_grad with the term attached = orc_score_grad without it + w_MDN * orc_mdn_energy at the same coordinates,
    for the energy, the per-atom gradient and (through the same chain rule) all 6+T pose components."""
    rec = synth.receptor(150, 15.0, 8, seed=1, grid_n=41, pocket_radius=4.0)
    radius, role = synth.type_table(8)
    ty, p = orc.Types(radius, role), orc.default_params()
    G = orc.build_grid(p, ty, rec.xyz, rec.type, rec.origin, rec.dims, rec.spacing)
    batch = synth.ligands([14], [3], 8, seed=5)
    L = orc.ligand_from_batch(batch, 0)
    order, res_off = synth.residues(rec, 8)
    rxyz = rec.xyz[order].astype(np.float64)
    pi, mu, sg = synth.gmm_params(len(res_off) - 1, L.n, 3, seed=9)
    pose = synth.random_poses(batch, [0], rec, seed=4, spread=0.4)[0, :7 + L.T].astype(np.float64)
    e0, g0, x0, ga0 = orc.score_grad(p, ty, G, L, pose)
    for w in (1.0, 0.37):
        L.set_mdn(orc.Mdn(rxyz, res_off, pi, mu, sg, w_mdn=w))
        e1, g1, x1, ga1 = orc.score_grad(p, ty, G, L, pose)
        Em, gm, _ = orc.mdn_energy(rxyz, res_off, pi, mu, sg, x0)
        assert Em < -0.05                                                      # the term is really there
        assert np.array_equal(x1, x0)
        assert e1[0] == pytest.approx(e0[0] + w * Em, rel=1e-13) and e1[1] == pytest.approx(e0[1] + w * Em, rel=1e-13)
        assert e1[2] == e0[2]
        assert np.allclose(ga1, ga0 + w * gm, rtol=1e-12, atol=1e-13)
        # pose gradient: central differences of the full energy on all 6+T components
        h = 1e-6
        E = lambda q: orc.score_grad(p, ty, G, L, q, want_grad=False)[0][0]
        for c in range(3):
            d = np.zeros_like(pose); d[c] = h
            assert g1[c] == pytest.approx((E(pose + d) - E(pose - d)) / (2 * h), rel=1e-5, abs=2e-5)
        for k in range(L.T):
            d = np.zeros_like(pose); d[7 + k] = h
            assert g1[6 + k] == pytest.approx((E(pose + d) - E(pose - d)) / (2 * h), rel=1e-5, abs=2e-5)
    L.set_mdn(None)
    assert orc.score_grad(p, ty, G, L, pose)[0][0] == e0[0]
    # hand case: one receptor atom = one residue at the origin, one ligand atom at distance 3 on the x axis, K = 1
    one = lambda v: np.array([[[v]]], dtype=np.float64)
    Em, gm, dm = orc.mdn_energy(np.zeros((1, 3)), np.array([0, 1]), one(1.0), one(3.0), one(0.5), np.array([[3.0, 0, 0]]))
    assert Em == pytest.approx(-1.0 / (0.5 * np.sqrt(2 * np.pi)), rel=1e-14) and gm[0, 0] == 0.0


def test_direct_receptor_mode_of_the_step_equals_the_direct_sums(orc):
    """NEXT-3: orc_score_grad handed a DirectReceptor = orc_score_grad_direct (itself pinned against the grid at nodes, the brute
    force field and central differences); an MC step under it moves downhill in the DIRECT energy."""
    rec = synth.receptor(150, 15.0, 8, seed=1, grid_n=41, pocket_radius=4.0)
    radius, role = synth.type_table(8)
    ty, p = orc.Types(radius, role), orc.default_params()
    batch = synth.ligands([14], [3], 8, seed=5)
    L = orc.ligand_from_batch(batch, 0)
    D = orc.DirectReceptor(rec.xyz, rec.type, 8)
    rng = np.random.default_rng(2)
    for s in range(4):
        pose = synth.random_poses(batch, [0], rec, seed=40 + s, spread=0.5)[0, :7 + L.T].astype(np.float64)
        e1, g1, x1, ga1 = orc.score_grad(p, ty, D, L, pose)
        e2, g2, x2, ga2 = orc.score_grad_direct(p, ty, rec.xyz, rec.type, L, pose)
        assert np.array_equal(e1, e2) and np.array_equal(g1, g2) and np.array_equal(ga1, ga2)
    # one accepted Adam step (tiny lr, no perturbation amplitude): first-order descent in the direct energy
    p2 = orc.default_params(lr=1e-5, pert_trans=0.0, pert_rot=0.0)
    for chain in range(40):
        u = orc.uniform4(7, chain, 0, 0, 0)
        if int(u[0] * (L.T + 2)) <= 1:
            break
    e0, g0, _, _ = orc.score_grad(p2, ty, D, L, pose)
    new, e_new, rec_ = orc.mc_step(p2, ty, D, L, 7, chain, 0, 0, rec.box_min, rec.box_max, pose, 1e9)
    assert rec_.accept == 1
    assert e_new - e0[0] == pytest.approx(-1e-5 * np.abs(g0).sum(), rel=2e-3)
