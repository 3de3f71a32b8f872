#!/usr/bin/env python
"""bench.py -- throughput of the tridsk hot path on synthetic workloads shaped like BASELINE.json's configs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--no-extras] [--impl reference]

A "step" is one pass of the whole hot path over one batch: receptor grid precompute (a0) + chain init, K_mc
fused MC steps for every chain of every ligand, top-k (a1..a10).  The default workload is C5, the largest
single-GPU configuration of BASELINE.json (its metric is quoted on no particular config).
`value` = score+grad pose evaluations per second of the whole job with inputs resident in HBM (chains x MC steps x
n_refine per second; `pose_evals_per_s` counts every FK+score evaluation, i.e. also the energy-only Metropolis
evaluation of each step and the initial one); `e2e` = the same through the C-ABI with HOST buffers (receptor + ligand
batch H2D, result D2H inside the timed region).  One JSON line on stdout (rank 0).
DESIGN.md section 7 states the accounting (evaluations, algorithmic FLOPs, the three roofline denominators).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import synth  # noqa: E402

METRIC = "score+grad pose evals/sec per B200"
UNIT = "score+grad pose evals/s"
KERNEL_NAMES = {1: "mc_kernel<J> (warp per chain)", 2: "mc_lane_kernel (lane per chain)", 3: "mc_cta_kernel (CTA per chain)",
                4: "mc_lane_tm_kernel (lane per chain, TMEM)"}
REGIME = {"C1": "latency", "C2": "latency", "C3": "throughput", "C4": "throughput", "C5": "throughput", "C2x32": "throughput",
          "P1": "latency", "M3": "throughput", "D2": "latency", "M2": "latency"}
MB_FFMA, MB_FFMA2, MB_MUFU, MB_L2_READ, MB_GATHER = range(5)


# ----------------------------------------------------------------------------------------- accounting
def work_of(n_atoms, n_tor, n_pairs, n_chains, n_steps, n_refine, mdn=None, direct=None):
    """Evaluations and ALGORITHMIC work of one step of a workload.  Two kinds of evaluation:
    G = score gradient (what an Adam step needs: FK, trilinear value + gradient, pair forces, reverse pass) and
    E = energy only (the Metropolis evaluation of a step, and the initial one).  Per MC step and chain: n_refine G
    evaluations, n_refine Adam updates, one E evaluation.  FMA = 2 flops."""
    n, t, p = (np.asarray(v, np.float64) for v in (n_atoms, n_tor, n_pairs))
    d = 6 + t
    flop_g = 28 * p + 116 * n + 140 * t        # pair: distance 8, Gaussian + derivative 8, clash 2, force 10; atom: trilinear 80, FK 21, reverse 15
    flop_e = 16 * p + 66 * n + 110 * t         # pair: distance 8, Gaussian 5, clash 3; atom: trilinear value 45, FK 21
    flop_adam = 20 * d
    xu_g, xu_e, xu_step = 2.0 * p, 2.3 * p, 2 * d + 10
    bytes_eval = 32 * n                        # 8 fp32 grid corners per atom per evaluation
    if mdn:                                    # E_MDN: per (atom, residue within the cut-off): minimum over the residue's atoms (8 flop each),
        hits, size, K = mdn["hits_per_atom"], mdn["res_size"], mdn["K"]            # then K Gaussians (value 8 flop, + derivative 4) and one sqrt
        flop_g = flop_g + n * hits * (8 * size + 12 * K + 8)
        flop_e = flop_e + n * hits * (8 * size + 8 * K)
        xu_g, xu_e = xu_g + n * hits * (K + 1), xu_e + n * hits * (K + 1)
        bytes_eval = bytes_eval + n * hits * (12 * K + 16 * size)   # three fp32 parameters per component, 16-byte atom records
    if direct:                                 # receptor term by direct sums: pairs within the range per atom instead of the trilinear lookup
        ppa = direct["pairs_per_atom"]
        flop_g = flop_g + n * (28 * ppa - 80)
        flop_e = flop_e + n * (16 * ppa - 45)
        xu_g, xu_e = xu_g + 2.0 * n * ppa, xu_e + 2.3 * n * ppa
        bytes_eval = 16 * n * ppa
    g_per_chain = n_steps * n_refine
    e_per_chain = n_steps + 1
    per_chain_flop = g_per_chain * (flop_g + flop_adam) + e_per_chain * flop_e
    per_chain_xu = g_per_chain * xu_g + e_per_chain * xu_e + n_steps * xu_step
    per_chain_bytes = (g_per_chain + e_per_chain) * bytes_eval
    ones = np.ones_like(n)
    return dict(evals=float(np.sum(n_chains * (g_per_chain + e_per_chain) * ones)), sg_evals=float(np.sum(n_chains * g_per_chain * ones)),
                flop=float(np.sum(n_chains * per_chain_flop)), xu=float(np.sum(n_chains * per_chain_xu)),
                gather_bytes=float(np.sum(n_chains * per_chain_bytes)))


_PEAKS = None


def peaks(eng=None, grid_bytes=None):
    """The three roofline denominators: derived from unit counts x clock, and measured on this device
    by the library's microbenchmarks (csrc/microbench.cu) in this process."""
    global _PEAKS
    sm_mhz, src, hbm = 1965.0, "fallback 1965 MHz (B200_PROFILING.md)", 6650.0
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        m = json.load(open(path))
        sm_mhz, hbm, src = float(m.get("sm_max_mhz", sm_mhz)), float(m.get("hbm_gbs", hbm)), "MEASURED_PEAKS.json sm_max_mhz"
    out = dict(alu_tflops=148 * 128 * 2 * sm_mhz * 1e6 / 1e12, xu_gops=148 * 16 * sm_mhz * 1e6 / 1e9, hbm_gbs=hbm, sm_mhz=sm_mhz,
               source=src)
    if eng is None:
        return out
    if _PEAKS is None:
        def rate(which, nbytes=0, iters=1, reps=3):
            best = 0.0
            for _ in range(reps):
                ms, work = eng.microbench(which, nbytes, iters)
                best = max(best, work / (ms * 1e-3))
            return best
        _PEAKS = dict(ffma_tflops=rate(MB_FFMA, 0, 2000) / 1e12, ffma2_tflops=rate(MB_FFMA2, 0, 2000) / 1e12,
                      mufu_gops=rate(MB_MUFU, 0, 1000) / 1e9,
                      l2_read_gbs=rate(MB_L2_READ, 33 << 20, 40) / 1e9,            # 33 MB: L2-resident streaming read
                      l2_gather_resident_gbs=rate(MB_GATHER, 33 << 20, 400) / 1e9)  # random sectors of an L2-resident buffer
    out.update(_PEAKS)
    if grid_bytes:
        ms, work = eng.microbench(MB_GATHER, int(grid_bytes), 400)
        out["gather_grid_gbs"] = work / (ms * 1e-3) / 1e9                           # random sectors of a buffer of the cell-packed grid's size
        out["gather_grid_bytes"] = int(grid_bytes)
    return out


def roofline_of(w, mc_ms, pk, kernel, traffic=None):
    """Times the three candidate bounds would need for the step's algorithmic work; the largest is the binding one."""
    t = mc_ms * 1e-3
    t_alu = w["flop"] / (pk["alu_tflops"] * 1e12)
    t_xu = w["xu"] / (pk["xu_gops"] * 1e9)
    l2_peak = pk.get("l2_read_gbs")
    t_l2 = w["gather_bytes"] / (l2_peak * 1e9) if l2_peak else 0.0
    bound = max((("alu", t_alu), ("xu", t_xu), ("l2", t_l2)), key=lambda kv: kv[1])[0]
    r = dict(bound=bound, kernel=kernel + ", fused MC step series",
             alu_frac=t_alu / t, xu_frac=t_xu / t, l2_frac=t_l2 / t,
             alu_tflops=w["flop"] / t / 1e12, xu_gops=w["xu"] / t / 1e9, grid_gather_gbs=w["gather_bytes"] / t / 1e9,
             traffic=traffic)
    if bound == "alu":
        r.update(achieved=r["alu_tflops"], peak=pk["alu_tflops"], unit="TFLOP/s", frac=r["alu_frac"])
    elif bound == "xu":
        r.update(achieved=r["xu_gops"], peak=pk["xu_gops"], unit="Gop/s", frac=r["xu_frac"])
    else:
        r.update(achieved=r["grid_gather_gbs"], peak=l2_peak, unit="GB/s", frac=r["l2_frac"])
    r["peaks"] = {k: pk[k] for k in pk if k not in ("source",)}
    r["peak_source"] = (f"alu: 148 SM x 128 lanes x 2 x {pk['sm_mhz']:.0f} MHz ({pk['source']}), measured FFMA stream "
                        f"{pk.get('ffma_tflops', float('nan')):.1f} / packed f32x2 {pk.get('ffma2_tflops', float('nan')):.1f} TFLOP/s; "
                        f"xu: 148 x 16 lanes x clock, measured ex2 stream {pk.get('mufu_gops', float('nan')):.0f} Gop/s; "
                        f"l2: measured streaming read of an L2-resident 33 MB buffer (csrc/microbench.cu, this run)")
    return r


def stored_traffic(name):
    """dram__bytes_read.sum + dram__bytes_write.sum of the MC kernel series of one step, from the ncu --set full capture
    summarised under profiles/ (profiles/r2_traffic.csv, written with the command that made it; never typed in here)."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    if not os.path.exists(path):
        return None
    for line in open(path):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 3 and f[0] == name:
            try:
                return float(f[2])
            except ValueError:
                return None
    return None


# ----------------------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.split(",") for r in open(self.f.name).read().strip().splitlines() if r.count(",") >= 6]
        os.unlink(self.f.name)
        if not rows:
            return out
        try:
            sm = [float(r[0]) for r in rows]
            busy = [s for s, r in zip(sm, rows) if float(r[2]) > 250.0] or sm       # samples under load
            out.update(sm_mhz=float(np.median(busy)), sm_max_mhz=float(rows[0][1]), samples=len(rows),
                       power_w_max=max(float(r[2]) for r in rows))
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            out["reasons"] = [n for i, n in enumerate(names) if any("Active" in r[3 + i] and "Not" not in r[3 + i] for r in rows)]
        except ValueError:
            pass
        return out


# ----------------------------------------------------------------------------------------- GPU arm
def run_workload(eng, name, steps, warmup, rank=0, world=1, do_e2e=True, sample_clocks=True, n_lig=None):
    import torch
    from paper_2510_24186_b200 import default_params, shard

    cfg = synth.CONFIGS[name]
    gp = default_params()
    gp.n_refine = cfg.n_refine
    rec = synth.make_receptor(cfg)
    radius, role = synth.type_table(cfg.n_types)
    batch_all = synth.make_ligands(cfg, n_lig)
    # multi-GPU: screens shard by ligand; single docks shard their chains (disjoint Philox chain ids)
    chain_base, n_chains, mine = 0, cfg.n_chains, None
    if batch_all.n_lig >= world and batch_all.n_lig > 1:
        mine = shard.ligand_shard(batch_all.n_lig, rank, world)
        batch = batch_all.subset(mine) if world > 1 else batch_all
        scaling = "strong"
    else:
        # weak scaling of a single dock: every rank runs the config's n_chains chains of its own (global ids rank * n_chains ..)
        batch, chain_base, scaling = batch_all, rank * cfg.n_chains, "weak"
    stride = 7 + int(np.max(np.diff(batch_all.tor_off)))
    d_xyz = torch.from_numpy(rec.xyz).to(eng.device)
    d_typ = torch.from_numpy(rec.type).to(eng.device)
    ligs = eng.load_ligands(batch, radius, role)
    mdn = None
    if cfg.mdn_K:                                                            # the paper's full score: attach E_MDN (synthetic parameters)
        res_xyz, res_off = synth.pocket_residues(rec)
        pi, mu, sg = synth.gmm_batch(len(res_off) - 1, np.diff(batch.atom_off), cfg.mdn_K, seed=cfg.lig_seed + 50000)
        eng.load_mdn(ligs, res_xyz, res_off, pi, mu, sg, cfg.mdn_K)
        mdn_host = (res_xyz, res_off, pi, mu, sg) if do_e2e else None       # the end-to-end leg attaches the term again
        del pi, mu, sg
        mdn = dict(K=cfg.mdn_K, n_res=len(res_off) - 1, res_size=float(np.mean(np.diff(res_off))))
    w = work_of(np.diff(batch.atom_off), np.diff(batch.tor_off), ligs.n_pairs, n_chains, cfg.n_steps, gp.n_refine)   # evaluation counts
    dock_kw = dict(receptor_direct=True) if cfg.direct else {}
    L, k = ligs.n_lig, cfg.top_k
    out = (torch.empty(L, k, 2, device=eng.device), torch.empty(L, k, stride, device=eng.device),
           torch.empty(L, k, dtype=torch.int32, device=eng.device))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=eng.device)     # > 126 MB L2
    dock_args = (gp, rec.box_min, rec.box_max, rec.pocket_center, rec.pocket_radius, n_chains, cfg.n_steps, k)

    def merge():
        """The one exchange of the multi-GPU path: every rank ends up with the complete result."""
        if world == 1:
            return out
        if scaling == "strong":
            return shard.merge_ligand_shards(out[0], out[1], out[2], batch_all.n_lig)
        return shard.merge_chain_shards(out[0], out[1], out[2], chain_base, k)

    def step():
        grid = eng.build_grid(d_xyz, d_typ, radius, role, gp, rec.origin, rec.dims, rec.spacing)
        if cfg.direct:
            eng.attach_receptor(grid, d_xyz, d_typ, radius, role, gp)
        eng.dock(grid, ligs, *dock_args, seed=cfg.philox_seed, pose_stride=stride, out=out, chain_base=chain_base, **dock_kw)
        merge()
        return grid

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step().free()
    barrier()
    sampler = ClockSampler(eng.device.index or 0) if sample_clocks else None
    launches0 = eng.launch_count()
    t_step, t_grid, t_mc, t_topk = [], [], [], []
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    wall0 = time.perf_counter()
    merged = out
    for _ in range(steps):
        with torch.cuda.stream(eng.stream):
            flush.zero_()                                                    # L2 flush, outside the timed events
            ev[0].record(eng.stream)
            grid = eng.build_grid(d_xyz, d_typ, radius, role, gp, rec.origin, rec.dims, rec.spacing)
            if cfg.direct:
                eng.attach_receptor(grid, d_xyz, d_typ, radius, role, gp)
            ev[1].record(eng.stream)
            eng.dock(grid, ligs, *dock_args, seed=cfg.philox_seed, pose_stride=stride, out=out, chain_base=chain_base, **dock_kw)
            merged = merge()
            ev[2].record(eng.stream)
        ev[2].synchronize()
        mc, tk = eng.last_dock_ms()
        t_grid.append(ev[0].elapsed_time(ev[1])); t_step.append(ev[0].elapsed_time(ev[2]))
        t_mc.append(mc); t_topk.append(tk)
        grid.free()
    barrier()
    wall = time.perf_counter() - wall0
    launches = eng.launch_count() - launches0
    clocks = sampler.stop() if sampler else {}
    ms = float(np.mean(t_step))
    if world > 1:
        tt = torch.tensor([ms], device=eng.device)
        torch.distributed.all_reduce(tt, op=torch.distributed.ReduceOp.MAX)
        ms = float(tt[0])
        tot = torch.tensor([w["evals"], w["sg_evals"]], device=eng.device, dtype=torch.float64)
        torch.distributed.all_reduce(tot)
        evals_all, sg_all = float(tot[0]), float(tot[1])
    else:
        evals_all, sg_all = w["evals"], w["sg_evals"]
    if mdn:                                                                  # (atom, residue) pairs inside the cut-off: counted on returned poses
        sample = list(range(0, L, max(1, L // 48)))[:48]
        li = np.asarray(sample, np.int32)
        poses = out[1][li, 0, :].contiguous().cpu().numpy()
        gtmp = eng.build_grid(d_xyz, d_typ, radius, role, gp, rec.origin, rec.dims, rec.spacing)
        _, _, xs = eng.score_grad(gtmp, ligs, gp, li, poses, want_grad=False)
        gtmp.free()
        hits = atoms = 0
        for q, l in enumerate(sample):
            nl = batch.n_atoms(l)
            dmat = np.linalg.norm(xs[q, :nl, None, :] - res_xyz[None, :, :], axis=2)             # [atom][receptor atom]
            dres = np.minimum.reduceat(dmat, res_off[:-1], axis=1)
            hits += int((dres < 5.0).sum()); atoms += nl
        mdn["hits_per_atom"] = hits / max(atoms, 1)
        w = work_of(np.diff(batch.atom_off), np.diff(batch.tor_off), ligs.n_pairs, n_chains, cfg.n_steps, gp.n_refine, mdn)
    direct = None
    if cfg.direct:                                                           # receptor atoms inside the pair function's range, per ligand atom
        li = np.zeros(1, np.int32)
        gtmp = eng.build_grid(d_xyz, d_typ, radius, role, gp, rec.origin, rec.dims, rec.spacing)
        _, _, xs = eng.score_grad(gtmp, ligs, gp, li, out[1][0, :1, :].contiguous().cpu().numpy(), want_grad=False)
        gtmp.free()
        nl = batch.n_atoms(0)
        dmat = np.linalg.norm(xs[0, :nl, None, :] - rec.xyz[None, :, :], axis=2)
        direct = dict(pairs_per_atom=float((dmat < gp.long_dmax).sum() / nl))
        w = work_of(np.diff(batch.atom_off), np.diff(batch.tor_off), ligs.n_pairs, n_chains, cfg.n_steps, gp.n_refine, None, direct)
    grid_bytes = 32 * int(np.prod(rec.dims)) * cfg.n_types                  # the cell-packed copy the kernels gather from (32 B per node)
    pk = peaks(eng, grid_bytes)
    mc_ms = float(np.mean(t_mc))
    res = dict(
        workload=name, title=cfg.title, n_lig=L, n_lig_all=batch_all.n_lig, n_chains=n_chains, n_steps=cfg.n_steps, top_k=k,
        evals=evals_all, sg_evals=sg_all, value=sg_all / (ms * 1e-3), pose_evals_per_s=evals_all / (ms * 1e-3),
        ms_per_step=ms, ms_per_task=ms / max(batch_all.n_lig, 1),
        ms_grid_build=float(np.mean(t_grid)), ms_mc_kernels=mc_ms, ms_topk=float(np.mean(t_topk)),
        wall_s=wall, launches=launches, scaling=scaling, clocks=clocks,
        roofline=roofline_of(w, mc_ms, pk, KERNEL_NAMES.get(eng.last_kernel(), "?"), stored_traffic(name) if n_lig is None and world == 1 else None),
        best_energy=float(merged[0][:, 0, 0].min().item()))
    res["roofline"]["mc_kernel_pose_evals_per_s"] = w["evals"] / (mc_ms * 1e-3)
    if mdn:
        res["mdn"] = mdn
    if direct:
        res["direct"] = direct
    if do_e2e:                                                               # host buffers in, host buffers out
        h_out = (np.empty((L, k, 2), np.float32), np.empty((L, k, stride), np.float32), np.empty((L, k), np.int32))
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
        h_xyz, h_typ = pin(rec.xyz), pin(rec.type)

        one_call = not cfg.mdn_K and not cfg.direct and chain_base == 0       # tridsk_screen: load + dock + free, packing overlapped

        def e2e_step():
            grid = eng.build_grid(h_xyz, h_typ, radius, role, gp, rec.origin, rec.dims, rec.spacing)
            if cfg.direct:
                eng.attach_receptor(grid, h_xyz, h_typ, radius, role, gp)
            if one_call:
                eng.screen(grid, batch, radius, role, *dock_args, seed=cfg.philox_seed, pose_stride=stride, out=h_out)
            else:
                lg = eng.load_ligands(batch, radius, role)
                if cfg.mdn_K:
                    eng.load_mdn(lg, *mdn_host, cfg.mdn_K)
                eng.dock(grid, lg, *dock_args, seed=cfg.philox_seed, pose_stride=stride, out=h_out, chain_base=chain_base, **dock_kw)
                lg.free()
            grid.free()
        e2e_step()                                                           # two untimed passes: the first one also pays first-touch
        e2e_step()                                                           # costs (pinned staging, allocator arenas, graph instantiation)
        barrier()
        n_e2e = max(1, min(steps, 5))
        passes = []
        for _ in range(n_e2e):                                               # every pass ends synchronised (host outputs)
            ts = time.perf_counter()
            e2e_step()
            passes.append(time.perf_counter() - ts)
        barrier()
        # the MEDIAN pass: a pass is one host-side packing + allocation + upload besides the GPU work, and on a shared host one in
        # a few passes takes 10-25 % longer (all pass times are in the line)
        e2e_s = float(np.median(passes))
        if world > 1:
            tt = torch.tensor([e2e_s], device=eng.device)
            torch.distributed.all_reduce(tt, op=torch.distributed.ReduceOp.MAX)
            e2e_s = float(tt[0])
        h2d = rec.xyz.nbytes + rec.type.nbytes + sum(getattr(batch, f).nbytes for f in (
            "atom_off", "ref_xyz", "atom_type", "atom_frag", "tor_off", "tor_a", "tor_b", "tor_parent", "bond_off", "bond_ab"))
        if cfg.mdn_K:
            h2d += sum(np.asarray(a).nbytes for a in mdn_host)
        res["e2e"] = dict(value=sg_all / e2e_s, unit=UNIT, h2d_bytes_per_step=int(h2d),
                          d2h_bytes_per_step=int(sum(a.nbytes for a in h_out)), ms_per_step=e2e_s * 1e3, steps=n_e2e,
                          statistic="median pass", ms_passes=[round(1e3 * t, 1) for t in passes], ms_mean=1e3 * float(np.mean(passes)),
                          note=("tridsk_build_grid + tridsk_screen (host packing of the batch, upload, dock, results to host buffers; the packing of most "
                                "of the batch overlaps the docking of its first part)" if one_call else
                                "tridsk_load_ligands (host packing of the batch + upload)" + (" + tridsk_load_mdn" if cfg.mdn_K else "") +
                                " + tridsk_build_grid + tridsk_dock with host buffers"))
        assert np.array_equal(h_out[2], out[2].cpu().numpy()), "e2e and device-resident legs disagree"
    ligs.free()
    return res


def run_multi_receptor(eng, n_targets=8, n_lig=256, n_chains=64, n_steps=100):
    """Many-target screen (DEKOIS 2.0 has 81 targets): n_targets receptors (C3-shaped, 3000 atoms, 80^3 x 16
    grid; every second one with 12 fixed waters), the same C3-shaped ligands docked to each, two passes over the targets through
    tridsk_build_grid_cached -- the second pass finds every grid in the per-receptor cache."""
    import torch
    from paper_2510_24186_b200 import default_params
    cfg = synth.CONFIGS["C3"]
    gp = default_params()
    radius, role = synth.type_table(cfg.n_types)
    batch = synth.make_ligands(cfg, n_lig)
    ligs = eng.load_ligands(batch, radius, role)
    stride = 7 + ligs.max_tor
    recs = []
    for t in range(n_targets):
        r = synth.receptor(cfg.n_rec, cfg.box_len, cfg.n_types, 1100 + t, cfg.grid_n)
        recs.append(synth.with_waters(r, 12, seed=t) if t % 2 else r)
    out = (torch.empty(n_lig, 1, 2, device=eng.device), torch.empty(n_lig, 1, stride, device=eng.device),
           torch.empty(n_lig, 1, dtype=torch.int32, device=eng.device))
    eng.grid_cache(budget_bytes=4 << 30)
    st0 = eng.grid_cache()
    t_pass = []
    for _ in range(2):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for r in recs:
            g = eng.build_grid_cached(r.xyz, r.type, radius, role, gp, r.origin, r.dims, r.spacing)
            eng.dock(g, ligs, gp, r.box_min, r.box_max, r.pocket_center, r.pocket_radius, n_chains, n_steps, 1, seed=0, pose_stride=stride, out=out)
            g.free()
        torch.cuda.synchronize()
        t_pass.append((time.perf_counter() - t0) * 1e3)
    st = eng.grid_cache()
    eng.grid_cache(budget_bytes=0)                                           # drop the grids
    eng.grid_cache(budget_bytes=4 << 30)
    ligs.free()
    sg = n_targets * n_lig * n_chains * n_steps
    return dict(title=f"{n_targets} receptors x {n_lig} ligands, two passes through the grid cache", ms_first_pass=t_pass[0], ms_second_pass=t_pass[1],
                value=sg / (t_pass[1] * 1e-3), unit=UNIT, cache_hits=st["hits"] - st0["hits"], cache_misses=st["misses"] - st0["misses"],
                cache_bytes=st["bytes"], regime="throughput", timing="host wall clock around each pass (grid builds + docks), synchronised")


# ----------------------------------------------------------------------------------------- oracle (CPU) arm
def _omp_threads(n):
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def oracle_sample(name, n_lig_sample, budget_s=12.0, grid=None, threads=None):
    """The oracle as it stands on the host cores, on a bounded sample of the workload: its grid build in full (once;
    the hot-path oracle reads a full grid), then the dock of the first n_lig_sample ligands -- all chains, as many MC steps
    as fit the time budget (the per-step cost of a chain does not depend on the step index)."""
    from oracle import oracle as orc
    cores = os.cpu_count() or 1
    cfg = synth.CONFIGS[name]
    rec = synth.make_receptor(cfg)
    radius, role = synth.type_table(cfg.n_types)
    batch = synth.make_ligands(cfg, min(n_lig_sample, cfg.n_lig))
    p = orc.default_params()
    p.n_refine = cfg.n_refine
    ty = orc.Types(radius, role)
    if threads:
        _omp_threads(threads)
    t0 = time.perf_counter()
    G = grid or orc.build_grid(p, ty, rec.xyz, rec.type, rec.origin, rec.dims, rec.spacing)
    t_grid = time.perf_counter() - t0
    Ls = [orc.ligand_from_batch(batch, i) for i in range(batch.n_lig)]

    def dock(ligs, ns):
        t = time.perf_counter()
        for i in ligs:
            orc.dock(p, ty, G, Ls[i], cfg.philox_seed, i, cfg.n_chains, ns, rec.box_min, rec.box_max, rec.pocket_center, rec.pocket_radius)
        return time.perf_counter() - t
    per_lig_step = dock([0], 2) / 2                                          # probe (includes the initial evaluation: conservative)
    ns = int(budget_s / max(per_lig_step * batch.n_lig, 1e-9))
    if ns >= 4:
        n_used, ns = batch.n_lig, min(ns, cfg.n_steps)
    else:                                                                    # too slow for every sample ligand: fewer ligands, 4 steps
        n_used, ns = max(1, min(batch.n_lig, int(budget_s / (per_lig_step * 4)))), 4
    t_dock = dock(range(n_used), ns)
    evals = n_used * cfg.n_chains * (ns * (p.n_refine + 1) + 1)
    sg = n_used * cfg.n_chains * ns * p.n_refine
    if threads:
        _omp_threads(cores)
    return dict(G=G, cores=threads or cores, t_grid=t_grid, t_dock=t_dock, pose_evals_per_s=evals / t_dock, sg_evals_per_s=sg / t_dock,
                sample=f"{name}: first {n_used} of {cfg.n_lig} ligand(s), {cfg.n_chains} chains x {ns} of {cfg.n_steps} MC steps "
                       f"({t_dock:.1f} s of oracle dock on {threads or cores} thread(s)); oracle grid build in full: {t_grid:.1f} s")


def cpu_baseline(name, budget_s=12.0):
    """cpu_baseline of the JSON line: the oracle's sampling rate (dock only) on all cores and on one thread; its brute-force
    fp64 grid build is a separate field (it is a table fill, not sampling, and would dominate a whole-step figure)."""
    cfg = synth.CONFIGS[name]
    n_s = {"C3": 64, "C5": 256}.get(name, cfg.n_lig)
    r = oracle_sample(name, n_s, budget_s)
    r1 = oracle_sample(name, n_s, budget_s / 3, grid=r["G"], threads=1)
    return dict(value=r["sg_evals_per_s"], unit=UNIT, cores=r["cores"], kind="oracle", sample=r["sample"],
                pose_evals_per_s=r["pose_evals_per_s"], grid_build_s=r["t_grid"],
                one_thread=dict(value=r1["sg_evals_per_s"], pose_evals_per_s=r1["pose_evals_per_s"], sample=r1["sample"]),
                note="dock-only rate scaled linearly in ligands (they are independent); grid_build_s is reported beside it, not folded in")


def run_reference(args):
    """--impl reference: the fp64 oracle on the host cores; each step = a bounded sample of the workload."""
    name = args.workload
    cfg = synth.CONFIGS[name]
    n_s = {"C3": 64, "C5": 256}.get(name, cfg.n_lig)
    first = oracle_sample(name, n_s, budget_s=6.0)
    vals = [first]
    for _ in range(max(args.warmup - 1, 0) + args.steps):
        vals.append(oracle_sample(name, n_s, budget_s=6.0, grid=first["G"]))
    timed = vals[-args.steps:]
    rate = float(np.mean([v["sg_evals_per_s"] for v in timed]))
    sg_step = cfg.n_lig * cfg.n_chains * cfg.n_steps * cfg.n_refine
    t_step = first["t_grid"] + sg_step / rate
    value = sg_step / t_step
    idx = int(name[1]) - 1 if name[0] == "C" and name[1:].isdigit() else -1
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=t_step * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=f"{name} {cfg.title}" + (f" (BASELINE.json configs[{idx}])" if idx >= 0 else ""),
                            note="each timed step = the oracle dock of a bounded sample (cpu_baseline.sample); ms_per_step = measured full "
                                 "grid build + the sampled dock rate scaled linearly to the full step"),
                cpu_baseline=dict(value=value, unit=UNIT, kind="oracle", cores=first["cores"], sample=first["sample"],
                                  dock_only_value=rate, grid_build_s=first["t_grid"]),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


# ----------------------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C5", choices=sorted(synth.CONFIGS))
    ap.add_argument("--impl", default="tridsk", choices=["tridsk", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the other configs' short runs")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle cpu_baseline leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg")
    ap.add_argument("--n-lig", type=int, default=None, help="first n ligands of a screening config (profiling)")
    ap.add_argument("--mc-steps", type=int, default=None, help="override the config's MC steps per chain (profiling only)")
    ap.add_argument("--kernel", type=int, default=0, help="force a chain-to-thread mapping (tridsk_set_kernel); 0 = automatic")
    args = ap.parse_args()
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))

    if args.impl == "reference":
        if rank == 0:
            run_reference(args)
        return

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    from paper_2510_24186_b200 import Engine
    torch.cuda.set_device(local)
    if world > 1:
        torch.distributed.init_process_group("nccl", device_id=torch.device("cuda", local))
    eng = Engine(local)
    eng.set_kernel(args.kernel)
    if args.mc_steps:
        import dataclasses
        synth.CONFIGS[args.workload] = dataclasses.replace(synth.CONFIGS[args.workload], n_steps=args.mc_steps)
    args.warmup = max(args.warmup, 3)
    main_res = run_workload(eng, args.workload, args.steps, args.warmup, rank, world, do_e2e=not args.no_e2e, n_lig=args.n_lig)
    extras = {}
    if not args.no_extras and world == 1 and args.n_lig is None:
        for name in sorted(synth.CONFIGS):
            if name == args.workload:
                continue
            big = name in ("C3", "C5")
            r = run_workload(eng, name, 2 if big else 5, 3, do_e2e=False, sample_clocks=False)
            extras[name] = {k: r[k] for k in ("title", "evals", "sg_evals", "value", "pose_evals_per_s", "ms_per_step", "ms_per_task",
                                              "ms_grid_build", "ms_mc_kernels", "ms_topk", "launches", "best_energy")}
            rf = r["roofline"]
            for kx in ("mdn", "direct"):
                if kx in r:
                    extras[name][kx] = r[kx]
            extras[name].update(kernel=rf["kernel"], regime=REGIME.get(name, "?"), bound=rf["bound"], roofline_frac=rf["frac"],
                                alu_frac=rf["alu_frac"], xu_frac=rf["xu_frac"], l2_frac=rf["l2_frac"],
                                gather_grid_gbs=rf["peaks"].get("gather_grid_gbs"),
                                mc_kernel_pose_evals_per_s=rf["mc_kernel_pose_evals_per_s"])
        extras["R8"] = run_multi_receptor(eng)
    if rank != 0:
        if world > 1:
            torch.distributed.destroy_process_group()
        return
    cfg = synth.CONFIGS[args.workload]
    cpu = None
    if not args.no_cpu and args.n_lig is None:
        cpu = cpu_baseline(args.workload)
    idx = int(args.workload[1]) - 1 if args.workload[0] == "C" and args.workload[1:].isdigit() else -1
    line = dict(
        metric=METRIC, value=main_res["value"], unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
        ms_per_step=main_res["ms_per_step"], higher_is_better=True, scaling=main_res["scaling"], vs_baseline=None,
        dtype="f32", data="synthetic",
        config=dict(workload=f"{args.workload} {cfg.title}" + (f" (BASELINE.json configs[{idx}], the largest single-GPU configuration)" if idx == 4
                                                                 else f" (BASELINE.json configs[{idx}])" if idx >= 0 else " (not a BASELINE.json config)"),
                    regime=REGIME.get(args.workload, "?"),
                    n_ligands=main_res["n_lig_all"], n_chains=main_res["n_chains"] * (world if main_res["scaling"] == "weak" else 1),
                    n_mc_steps=cfg.n_steps, top_k=cfg.top_k, n_refine=cfg.n_refine,
                    l2="flushed between steps (256 MiB memset outside the timed events)",
                    step="grid build (a0) + init + MC steps + top-k (a1..a10), one CUDA-graph launch" + (" + shard merge (all_gather)" if world > 1 else "")),
        pose_evals_per_s=main_res["pose_evals_per_s"], ms_per_task=main_res["ms_per_task"],
        ms_grid_build=main_res["ms_grid_build"], ms_mc_kernels=main_res["ms_mc_kernels"], ms_topk=main_res["ms_topk"],
        clocks=main_res["clocks"], e2e=main_res.get("e2e"), gpu_launches=main_res["launches"],
        roofline=main_res["roofline"], mdn=main_res.get("mdn"), cpu_baseline=cpu, best_energy=main_res["best_energy"], other_workloads=extras)
    print(json.dumps(line))
    eng.close()
    if world > 1:
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
