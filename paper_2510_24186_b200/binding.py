"""Thin ctypes binding over libtridsk.so (include/tridsk.h): argument marshalling only.

Every step of the path runs in the CUDA kernels; PyTorch is used for device memory and
streams, numpy for host buffers.  Buffers may be numpy arrays (host pointers) or CUDA torch
tensors (device pointers) -- the library detects which.  There is no CPU fallback: a missing
or unloadable extension raises at import of the first call.
"""
from __future__ import annotations

import ctypes as C
import os
import weakref

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtridsk.so")

OK, EINVAL, ENOMEM, ECUDA, ELIMIT = 0, -1, -2, -3, -4


class TridskError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"tridsk error {code}: {msg}")
        self.code = code


class Params(C.Structure):
    """tridsk_params (include/tridsk.h)."""
    _fields_ = [(n, C.c_float) for n in (
        "w_long", "w_clash", "w_hbond", "long_mu", "long_two_sigma2", "long_dmax",
        "hb_mu", "hb_sigma", "hb_dmax", "hb_dclash", "d_floor", "k_wall",
        "beta", "lr", "adam_b1", "adam_b2", "adam_eps", "pert_trans", "pert_rot", "w_tor")] + [("n_refine", C.c_int)]


class _Types(C.Structure):
    _fields_ = [("n_types", C.c_int), ("radius", C.c_void_p), ("hb_role", C.c_void_p)]


class _Batch(C.Structure):
    _fields_ = [("n_lig", C.c_int)] + [(n, C.c_void_p) for n in (
        "atom_off", "ref_xyz", "atom_type", "atom_frag", "tor_off", "tor_a", "tor_b", "tor_parent",
        "pair_off", "pair_ab", "bond_off", "bond_ab")]


class _Mdn(C.Structure):
    """tridsk_mdn (include/tridsk.h)."""
    _fields_ = [("n_res", C.c_int), ("res_off", C.c_void_p), ("res_xyz", C.c_void_p), ("K", C.c_int), ("pi", C.c_void_p),
                ("mu", C.c_void_p), ("sigma", C.c_void_p), ("w_mdn", C.c_float), ("d_cut", C.c_float)]


class _DockOpts(C.Structure):
    _fields_ = [("first_step", C.c_int), ("init_poses", C.c_void_p), ("resume", C.c_int),
                ("chain_state", C.c_void_p), ("trace", C.c_void_p), ("steps_per_launch", C.c_int),
                ("no_graph", C.c_int), ("chain_base", C.c_int), ("cluster_rmsd", C.c_float), ("receptor_direct", C.c_int),
                ("lig_base", C.c_int)]


TRACE_DTYPE = np.dtype([("e_prop", np.float32), ("e_cur", np.float32), ("u", np.float32), ("flags", np.int32)])

_lib = None


def lib():
    """Load libtridsk.so, (re)building it with nvcc first if it is missing or older than its sources (content-hash
    stamp); fails loudly if that is impossible -- there is no CPU fallback."""
    global _lib
    if _lib is None:
        try:
            from . import build as _build
            _build.build()
        except Exception as exc:                              # no nvcc, compile error, ...
            if not os.path.exists(LIB_PATH):
                raise ImportError(f"{LIB_PATH} is missing and could not be built ({exc}); build it with "
                                  "`python -m paper_2510_24186_b200.build` (there is no CPU fallback)") from exc
        _lib = C.CDLL(LIB_PATH)
        _lib.tridsk_last_error.restype = C.c_char_p
        _lib.tridsk_launch_count.restype = C.c_longlong
        _lib.tridsk_launch_count.argtypes = [C.c_void_p]
        _lib.tridsk_last_kernel.restype = C.c_int
        _lib.tridsk_last_kernel.argtypes = [C.c_void_p]
        _lib.tridsk_last_error.argtypes = [C.c_void_p]
        for name in ("tridsk_destroy", "tridsk_free_grid", "tridsk_free_ligands"):
            getattr(_lib, name).restype = None
            getattr(_lib, name).argtypes = [C.c_void_p]
    return _lib


def default_params(**kw) -> Params:
    p = Params()
    lib().tridsk_default_params(C.byref(p))
    for k, v in kw.items():
        setattr(p, k, v)
    return p


def _ptr(a):
    """Raw pointer of a numpy array (host) or a torch tensor (host or device); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return C.c_void_p(a.ctypes.data)
    assert a.is_contiguous()
    return C.c_void_p(a.data_ptr())


def _f3(v):
    return (C.c_float * 3)(*[float(x) for x in v])


class Grid:
    def __init__(self, eng, handle, n_types, dims, origin, spacing):
        self.eng, self.handle, self.n_types, self.dims = eng, handle, n_types, tuple(dims)
        self.origin, self.spacing = np.asarray(origin, np.float32), float(spacing)
        eng._children.add(self)

    def export(self):
        nx, ny, nz = self.dims
        out = np.empty((self.n_types, nz, ny, nx), np.float32)
        self.eng._ck(lib().tridsk_grid_export(self.eng.ctx, self.handle, _ptr(out)))
        return out

    def free(self):
        if self.handle:
            lib().tridsk_free_grid(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Ligands:
    def __init__(self, eng, handle):
        self.eng, self.handle = eng, handle
        eng._children.add(self)
        n, na, nt = C.c_int(), C.c_int(), C.c_int()
        lib().tridsk_ligand_info(handle, C.byref(n), C.byref(na), C.byref(nt), None)
        self.n_lig, self.max_atoms, self.max_tor = n.value, na.value, nt.value
        self.n_pairs = np.zeros(self.n_lig, np.int32)
        lib().tridsk_ligand_info(handle, None, None, None, _ptr(self.n_pairs))

    def free(self):
        if self.handle:
            lib().tridsk_free_ligands(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Engine:
    """One tridsk_ctx on one CUDA device, with its own torch stream."""

    def __init__(self, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("tridsk needs a CUDA device: there is no CPU fallback")
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.stream = torch.cuda.Stream(device=self.device)
        self.ctx = C.c_void_p()
        self._children = weakref.WeakSet()      # live Grid / Ligands handles: freed before the ctx
        rc = lib().tridsk_create(C.byref(self.ctx), C.c_int(device), C.c_void_p(self.stream.cuda_stream))
        if rc != OK:
            raise TridskError(rc, "tridsk_create failed")

    def _ck(self, rc):
        if rc != OK:
            raise TridskError(rc, lib().tridsk_last_error(self.ctx).decode())

    def close(self):
        for ch in list(self._children):
            ch.free()
        if self.ctx:
            lib().tridsk_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def synchronize(self):
        self._ck(lib().tridsk_synchronize(self.ctx))

    def set_kernel(self, kernel: int):
        """0 auto, 1 warp per chain, 2 lane per chain, 3 CTA per chain, 4 lane per chain with coordinates in tensor memory
        (tridsk_set_kernel)."""
        self._ck(lib().tridsk_set_kernel(self.ctx, C.c_int(kernel)))

    def last_kernel(self) -> int:
        """Mapping the last dock used: 1 warp, 2 lane, 3 CTA per chain (tridsk_last_kernel)."""
        return int(lib().tridsk_last_kernel(self.ctx))

    def launch_count(self) -> int:
        return int(lib().tridsk_launch_count(self.ctx))

    def _sync_in(self):
        """Order our stream after whatever torch has enqueued on its current stream."""
        self.stream.wait_stream(self.torch.cuda.current_stream(self.device))

    def _sync_out(self):
        self.torch.cuda.current_stream(self.device).wait_stream(self.stream)

    @staticmethod
    def _types(radius, role):
        radius = np.ascontiguousarray(radius, np.float32)
        role = np.ascontiguousarray(role, np.uint8)
        return _Types(len(radius), radius.ctypes.data, role.ctypes.data), (radius, role)

    # ------------------------------------------------------------------ grid
    def build_grid(self, rec_xyz, rec_type, radius, role, params, origin, dims, spacing) -> Grid:
        ty, keep = self._types(radius, role)
        if isinstance(rec_xyz, np.ndarray):
            rec_xyz = np.ascontiguousarray(rec_xyz, np.float32)
            rec_type = np.ascontiguousarray(rec_type, np.int32)
        n_rec = int(rec_xyz.shape[0])
        h = C.c_void_p()
        self._sync_in()
        self._ck(lib().tridsk_build_grid(self.ctx, _ptr(rec_xyz), _ptr(rec_type), C.c_int(n_rec), C.byref(ty),
                                         C.byref(params), _f3(origin), (C.c_int * 3)(*[int(d) for d in dims]),
                                         C.c_float(spacing), C.byref(h)))
        self._sync_out()
        return Grid(self, h, ty.n_types, dims, origin, spacing)

    def build_grid_cached(self, rec_xyz, rec_type, radius, role, params, origin, dims, spacing) -> Grid:
        """tridsk_build_grid_cached: the grid through the ctx's per-receptor cache (a hit launches nothing)."""
        ty, keep = self._types(radius, role)
        xyz = rec_xyz if not isinstance(rec_xyz, np.ndarray) else np.ascontiguousarray(rec_xyz, np.float32)
        typ = rec_type if not isinstance(rec_type, np.ndarray) else np.ascontiguousarray(rec_type, np.int32)
        h = C.c_void_p()
        d = (C.c_int * 3)(*[int(v) for v in dims])
        self._sync_in()
        self._ck(lib().tridsk_build_grid_cached(self.ctx, _ptr(xyz), _ptr(typ), C.c_int(int(xyz.shape[0])), C.byref(ty), C.byref(params),
                                                _f3(origin), d, C.c_float(spacing), C.byref(h)))
        self._sync_out()
        return Grid(self, h, ty.n_types, dims, origin, spacing)

    def attach_receptor(self, grid: Grid, rec_xyz, rec_type, radius, role, params):
        """tridsk_grid_attach_receptor: the receptor for dock(..., receptor_direct=True)."""
        ty, keep = self._types(radius, role)
        xyz = rec_xyz if not isinstance(rec_xyz, np.ndarray) else np.ascontiguousarray(rec_xyz, np.float32)
        typ = rec_type if not isinstance(rec_type, np.ndarray) else np.ascontiguousarray(rec_type, np.int32)
        self._sync_in()
        self._ck(lib().tridsk_grid_attach_receptor(self.ctx, grid.handle, _ptr(xyz), _ptr(typ), C.c_int(int(xyz.shape[0])), C.byref(ty),
                                                   C.byref(params)))

    def grid_cache(self, budget_bytes=-1):
        """Set the cache's byte budget (-1: leave it) -> dict(hits, misses, grids, bytes)."""
        st = (C.c_longlong * 4)()
        self._ck(lib().tridsk_grid_cache_config(self.ctx, C.c_longlong(int(budget_bytes)), st))
        return dict(hits=st[0], misses=st[1], grids=st[2], bytes=st[3])

    def grid_from_values(self, values, origin, spacing) -> Grid:
        if isinstance(values, np.ndarray):
            values = np.ascontiguousarray(values, np.float32)
        nt, nz, ny, nx = values.shape
        h = C.c_void_p()
        self._sync_in()
        self._ck(lib().tridsk_grid_from_values(self.ctx, _ptr(values), C.c_int(nt), _f3(origin),
                                               (C.c_int * 3)(nx, ny, nz), C.c_float(spacing), C.byref(h)))
        return Grid(self, h, nt, (nx, ny, nz), origin, spacing)

    # ------------------------------------------------------------------ ligands
    def load_ligands(self, batch, radius, role, pairs=None) -> Ligands:
        """batch: any object with the arrays of tridsk_ligand_batch (e.g. workloads.synth.LigandBatch).
        pairs: optional (pair_off, pair_ab); otherwise the library derives them from the bonds."""
        ty, keep = self._types(radius, role)
        b, arrs = self._batch(batch, pairs)
        h = C.c_void_p()
        self._ck(lib().tridsk_load_ligands(self.ctx, C.byref(b), C.byref(ty), C.byref(h)))
        return Ligands(self, h)

    @staticmethod
    def _batch(batch, pairs=None):
        """tridsk_ligand_batch over the arrays of `batch` (no copies when they already have the ABI's dtypes)."""
        A = lambda a, dt: np.ascontiguousarray(a, dt)
        arrs = dict(atom_off=A(batch.atom_off, np.int32), ref_xyz=A(batch.ref_xyz, np.float32),
                    atom_type=A(batch.atom_type, np.uint8), atom_frag=A(batch.atom_frag, np.uint8),
                    tor_off=A(batch.tor_off, np.int32), tor_a=A(batch.tor_a, np.uint8), tor_b=A(batch.tor_b, np.uint8),
                    tor_parent=A(batch.tor_parent, np.int8))
        if pairs is not None:
            arrs["pair_off"], arrs["pair_ab"] = A(pairs[0], np.int32), A(pairs[1], np.uint8)
        else:
            arrs["bond_off"], arrs["bond_ab"] = A(batch.bond_off, np.int32), A(batch.bond_ab, np.uint8)
        b = _Batch(n_lig=int(batch.n_lig))
        for k, v in arrs.items():
            setattr(b, k, v.ctypes.data)
        return b, arrs

    def screen(self, grid: Grid, batch, radius, role, params, box_min, box_max, pocket_center, pocket_radius,
               n_chains, n_steps, top_k, seed=0, pose_stride=None, out=None, pairs=None):
        """tridsk_screen: load + dock + free of a host ligand batch in one call (the packing of most of the batch overlaps the
        docking of its first part).  -> dict(energy[n_lig,k,2], pose[n_lig,k,stride], chain[n_lig,k]); `out`: optional
        pre-allocated buffers (numpy or CUDA tensors)."""
        ty, keep = self._types(radius, role)
        b, arrs = self._batch(batch, pairs)
        L = int(batch.n_lig)
        stride = int(pose_stride or (7 + int(np.max(np.diff(arrs["tor_off"])) if L else 0)))
        if out is not None:
            energy, pose, chain = out
        else:
            energy = np.empty((L, top_k, 2), np.float32)
            pose = np.empty((L, top_k, stride), np.float32)
            chain = np.empty((L, top_k), np.int32)
        self._sync_in()
        self._ck(lib().tridsk_screen(self.ctx, grid.handle, C.byref(b), C.byref(ty), C.byref(params), _f3(box_min), _f3(box_max),
                                     _f3(pocket_center), C.c_float(pocket_radius), C.c_int(n_chains), C.c_int(n_steps),
                                     C.c_int(top_k), C.c_ulonglong(seed), C.c_int(stride), _ptr(energy), _ptr(pose), _ptr(chain)))
        self._sync_out()
        return dict(energy=energy, pose=pose, chain=chain)

    def load_mdn(self, ligs: Ligands, res_xyz, res_off, pi, mu, sigma, K, w_mdn=1.0, d_cut=5.0):
        """Attach the mixture-density term (tridsk_load_mdn) to a ligand batch.  res_xyz [n_at,3], res_off [n_res+1]: host;
        pi, mu, sigma: flat float32 arrays (numpy, or torch tensors on the host or the device), ligand-major blocks
        [n_res][n_atoms(l)][K] in the caller's atom order."""
        A = lambda a, dt: np.ascontiguousarray(a, dt)
        xyz, off = A(res_xyz, np.float32), A(res_off, np.int32)
        par = [A(a, np.float32).reshape(-1) if isinstance(a, np.ndarray) else a.contiguous().reshape(-1) for a in (pi, mu, sigma)]
        m = _Mdn(len(off) - 1, off.ctypes.data, xyz.ctypes.data, int(K), _ptr(par[0]), _ptr(par[1]), _ptr(par[2]), float(w_mdn), float(d_cut))
        self._sync_in()
        self._ck(lib().tridsk_load_mdn(self.ctx, ligs.handle, C.byref(m)))

    def unload_mdn(self, ligs: Ligands):
        self._ck(lib().tridsk_load_mdn(self.ctx, ligs.handle, None))

    # ------------------------------------------------------------------ score + gradient
    def score_grad(self, grid: Grid, ligs: Ligands, params, lig_index, poses, want_grad=True, want_coords=True):
        """Host (numpy) or device (torch CUDA) in, same kind out.  -> energy[n,3], grad[n,6+Tmax], coords[n,Nmax,3]."""
        dev = not isinstance(poses, np.ndarray)
        n, stride = int(poses.shape[0]), int(poses.shape[1])
        gs, cs = 6 + ligs.max_tor, ligs.max_atoms
        if dev:
            t = self.torch
            mk = lambda *s: t.empty(*s, dtype=t.float32, device=self.device)
        else:
            poses = np.ascontiguousarray(poses, np.float32)
            lig_index = np.ascontiguousarray(lig_index, np.int32)
            mk = lambda *s: np.empty(s, np.float32)
        energy = mk(n, 3)
        grad = mk(n, gs) if want_grad else None
        coords = mk(n, cs, 3) if want_coords else None
        self._sync_in()
        self._ck(lib().tridsk_score_grad(self.ctx, grid.handle, ligs.handle, C.byref(params), _ptr(lig_index), _ptr(poses),
                                         C.c_int(n), C.c_int(stride), _ptr(energy), _ptr(grad), C.c_int(gs),
                                         _ptr(coords), C.c_int(cs)))
        self._sync_out()
        return energy, grad, coords

    def score_direct(self, rec_xyz, rec_type, radius, role, ligs: Ligands, params, lig_index, poses, want_grad=True):
        """tridsk_score_direct: receptor term as direct sums over the receptor atoms (no grid).  Host (numpy) buffers.
        -> energy[n,3], grad[n,6+Tmax]."""
        ty, keep = self._types(radius, role)
        rec_xyz = np.ascontiguousarray(rec_xyz, np.float32)
        rec_type = np.ascontiguousarray(rec_type, np.int32)
        poses = np.ascontiguousarray(poses, np.float32)
        lig_index = np.ascontiguousarray(lig_index, np.int32)
        n, stride, gs = int(poses.shape[0]), int(poses.shape[1]), 6 + ligs.max_tor
        energy = np.empty((n, 3), np.float32)
        grad = np.empty((n, gs), np.float32) if want_grad else None
        self._sync_in()
        self._ck(lib().tridsk_score_direct(self.ctx, _ptr(rec_xyz), _ptr(rec_type), C.c_int(int(rec_xyz.shape[0])), C.byref(ty),
                                           C.byref(params), ligs.handle, _ptr(lig_index), _ptr(poses), C.c_int(n), C.c_int(stride),
                                           _ptr(energy), _ptr(grad), C.c_int(gs)))
        self._sync_out()
        return energy, grad

    # ------------------------------------------------------------------ dock
    def dock(self, grid: Grid, ligs: Ligands, params, box_min, box_max, pocket_center, pocket_radius,
             n_chains, n_steps, top_k, seed=0, pose_stride=None, device_out=False, init_poses=None,
             first_step=0, resume=False, chain_state=None, want_state=False, want_trace=False,
             steps_per_launch=0, no_graph=False, chain_base=0, out=None, cluster_rmsd=0.0, receptor_direct=False, lig_base=0):
        """-> dict(energy[n_lig,k,2], pose[n_lig,k,stride], chain[n_lig,k], state?, trace?).
        device_out: outputs are CUDA torch tensors (no D2H, no sync); else numpy (D2H inside the call).
        out: optional pre-allocated (energy, pose, chain) buffers to write into."""
        t = self.torch
        stride = int(pose_stride or (7 + ligs.max_tor))
        L = ligs.n_lig
        if out is not None:
            energy, pose, chain = out
        elif device_out:
            energy = t.empty(L, top_k, 2, dtype=t.float32, device=self.device)
            pose = t.empty(L, top_k, stride, dtype=t.float32, device=self.device)
            chain = t.empty(L, top_k, dtype=t.int32, device=self.device)
        else:
            energy = np.empty((L, top_k, 2), np.float32)
            pose = np.empty((L, top_k, stride), np.float32)
            chain = np.empty((L, top_k), np.int32)
        o = _DockOpts()
        o.first_step, o.resume = int(first_step), int(bool(resume))
        o.steps_per_launch, o.no_graph = int(steps_per_launch), int(bool(no_graph))
        o.chain_base = int(chain_base)
        o.cluster_rmsd = float(cluster_rmsd)
        o.receptor_direct = int(bool(receptor_direct))
        o.lig_base = int(lig_base)
        keep = []
        if init_poses is not None:
            if isinstance(init_poses, np.ndarray):
                init_poses = np.ascontiguousarray(init_poses, np.float32)
            assert tuple(init_poses.shape) == (L, n_chains, stride)
            o.init_poses = _ptr(init_poses).value
            keep.append(init_poses)
        state = chain_state
        if state is None and (want_state or resume):
            state = np.zeros(L * n_chains * (2 * stride + 2), np.float32)
        if state is not None:
            o.chain_state = _ptr(state).value
        trace = None
        if want_trace:
            trace = np.zeros((L, n_chains, n_steps), TRACE_DTYPE)
            o.trace = _ptr(trace).value
        self._sync_in()
        self._ck(lib().tridsk_dock(self.ctx, grid.handle, ligs.handle, C.byref(params), _f3(box_min), _f3(box_max),
                                   _f3(pocket_center), C.c_float(pocket_radius), C.c_int(n_chains), C.c_int(n_steps),
                                   C.c_int(top_k), C.c_ulonglong(seed), C.c_int(stride), _ptr(energy), _ptr(pose),
                                   _ptr(chain), C.byref(o)))
        self._sync_out()
        res = dict(energy=energy, pose=pose, chain=chain)
        if state is not None:
            res["state"] = state
        if trace is not None:
            res["trace"] = trace
        return res

    def dock_static(self, grid: Grid, ligs: Ligands, params, box_min, box_max, pocket_center, pocket_radius,
                    n_chains, n_steps, top_k, out, seed=0, pose_stride=None):
        """tridsk_dock_static: the docking run without any allocation (chain state in the library's 4 MiB static device
        array); `out` = caller-allocated CUDA tensors (energy[n_lig,k,2], pose[n_lig,k,stride], chain[n_lig,k] int32)."""
        stride = int(pose_stride or (7 + ligs.max_tor))
        energy, pose, chain = out
        self._sync_in()
        self._ck(lib().tridsk_dock_static(self.ctx, grid.handle, ligs.handle, C.byref(params), _f3(box_min), _f3(box_max),
                                          _f3(pocket_center), C.c_float(pocket_radius), C.c_int(n_chains), C.c_int(n_steps),
                                          C.c_int(top_k), C.c_ulonglong(seed), C.c_int(stride), _ptr(energy), _ptr(pose),
                                          _ptr(chain)))
        self._sync_out()
        return dict(energy=energy, pose=pose, chain=chain)

    def last_dock_ms(self):
        """(MC kernel series, top-k) device milliseconds of the last dock, from CUDA events on the ctx stream."""
        ms = (C.c_float * 2)()
        self._ck(lib().tridsk_last_dock_ms(self.ctx, ms))
        return float(ms[0]), float(ms[1])

    def microbench(self, which, nbytes=0, iters=1):
        """One launch of a roofline microbenchmark (tridsk_debug_microbench): returns (ms, work)."""
        ms, work = C.c_float(), C.c_double()
        self._ck(lib().tridsk_debug_microbench(self.ctx, int(which), C.c_ulonglong(int(nbytes)), int(iters), C.byref(ms), C.byref(work)))
        return float(ms.value), float(work.value)

    def philox(self, ctr, key):
        out = (C.c_uint * 4)()
        self._ck(lib().tridsk_debug_philox(self.ctx, (C.c_uint * 4)(*ctr), (C.c_uint * 2)(*key), out))
        return list(out)


def split_state(state, n_lig, n_chains, stride):
    """Views of a chain_state buffer: pose_cur, pose_best [n_lig,n_chains,stride], e_cur, e_best [n_lig,n_chains]."""
    n = n_lig * n_chains
    pc = state[: n * stride].reshape(n_lig, n_chains, stride)
    pb = state[n * stride: 2 * n * stride].reshape(n_lig, n_chains, stride)
    ec = state[2 * n * stride: 2 * n * stride + n].reshape(n_lig, n_chains)
    eb = state[2 * n * stride + n: 2 * n * stride + 2 * n].reshape(n_lig, n_chains)
    return pc, pb, ec, eb
