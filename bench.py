#!/usr/bin/env python
"""bench.py -- throughput of the tridsk hot path on synthetic workloads shaped like BASELINE.json's configs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--no-extras] [--impl reference]

A "step" is one pass of the whole hot path over one batch: receptor grid precompute (a0) + chain init, K_mc
fused MC steps for every chain of every ligand, top-k (a1..a10).  `value` = FK+score pose evaluations per
second of the whole job with inputs resident in HBM; `e2e` = the same through the C-ABI with HOST buffers
(receptor + ligand H2D, result D2H inside the timed region).  One JSON line on stdout (rank 0).
DESIGN.md section 7 states the accounting (evaluations, algorithmic FLOPs, peaks).
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
UNIT = "pose evals/s"
KERNEL_NAMES = {1: "mc_kernel<J> (warp per chain)", 2: "mc_lane_kernel (lane per chain)", 3: "mc_cta_kernel (CTA per chain)"}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the `ncu --set full` captures
# summarised under profiles/ (r1b_ncu_full_cta_c2.txt, r1b_ncu_full_lane_c5.txt); None where no capture was made
NCU_TRAFFIC_BYTES = {"C2": 14.50e6}


# ----------------------------------------------------------------------------------------- accounting
def work_of(n_atoms, n_tor, n_pairs, n_chains, n_steps, n_refine):
    """Evaluations and algorithmic work (SURVEY.md 8(d) / DESIGN.md 7) of one step of a workload."""
    n, t, p = (np.asarray(v, np.float64) for v in (n_atoms, n_tor, n_pairs))
    evals_per_chain = n_steps * (n_refine + 1) + 1            # init + per MC step: n_refine score+grad + 1 score
    flop_per_eval = 30 * p + 116 * n + 140 * t + 20 * (6 + t)  # 30P + 80N + 36N + 140T + 20D
    xu_per_eval = 2.2 * p + 2 * (6 + t) + 10
    bytes_per_eval = 32 * n                                    # 8 fp32 grid corners per atom
    per_lig = n_chains * evals_per_chain
    return dict(evals=float(np.sum(per_lig * np.ones_like(n))), sg_evals=float(len(n) * n_chains * n_steps * n_refine),
                flop=float(np.sum(per_lig * flop_per_eval)), xu=float(np.sum(per_lig * xu_per_eval)),
                gather_bytes=float(np.sum(per_lig * bytes_per_eval)))


def peaks():
    sm_mhz, src = 1965.0, "fallback 1965 MHz (B200_PROFILING.md)"
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm = 6650.0
    if os.path.exists(path):
        m = json.load(open(path))
        sm_mhz, hbm, src = float(m.get("sm_max_mhz", sm_mhz)), float(m.get("hbm_gbs", hbm)), "MEASURED_PEAKS.json sm_max_mhz"
    # FP32 ALU peak: 148 SMs x 128 FP32 lanes x 2 flop (FMA) x max SM clock
    return dict(alu_tflops=148 * 128 * 2 * sm_mhz * 1e6 / 1e12, xu_gops=148 * 16 * sm_mhz * 1e6 / 1e9, hbm_gbs=hbm,
                sm_mhz=sm_mhz, source=src)


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
    from paper_2510_24186_b200 import default_params

    cfg = synth.CONFIGS[name]
    gp = default_params()
    gp.n_refine = cfg.n_refine
    rec = synth.make_receptor(cfg)
    radius, role = synth.type_table(cfg.n_types)
    batch_all = synth.make_ligands(cfg, n_lig)
    # multi-GPU: screens shard by ligand; single docks replicate the ligand with disjoint chain ids
    chain_base = 0
    if batch_all.n_lig >= world and batch_all.n_lig > 1:
        mine = list(range(rank, batch_all.n_lig, world))
        batch = batch_all.subset(mine) if world > 1 else batch_all
        scaling = "strong"
    else:
        batch, chain_base, scaling = batch_all, rank * cfg.n_chains, "weak"
    stride = 7 + int(np.max(np.diff(batch.tor_off)))
    d_xyz = torch.from_numpy(rec.xyz).to(eng.device)
    d_typ = torch.from_numpy(rec.type).to(eng.device)
    ligs = eng.load_ligands(batch, radius, role)
    w = work_of(np.diff(batch.atom_off), np.diff(batch.tor_off), ligs.n_pairs, cfg.n_chains, cfg.n_steps, gp.n_refine)
    L, k = ligs.n_lig, cfg.top_k
    out = (torch.empty(L, k, 2, device=eng.device), torch.empty(L, k, stride, device=eng.device),
           torch.empty(L, k, dtype=torch.int32, device=eng.device))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=eng.device)     # > 126 MB L2
    dock_args = (gp, rec.box_min, rec.box_max, rec.pocket_center, rec.pocket_radius, cfg.n_chains, cfg.n_steps, k)

    def step():
        grid = eng.build_grid(d_xyz, d_typ, radius, role, gp, rec.origin, rec.dims, rec.spacing)
        eng.dock(grid, ligs, *dock_args, seed=cfg.philox_seed, pose_stride=stride, out=out, chain_base=chain_base)
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
    for _ in range(steps):
        with torch.cuda.stream(eng.stream):
            flush.zero_()                                                    # L2 flush, outside the timed events
            ev[0].record(eng.stream)
            grid = eng.build_grid(d_xyz, d_typ, radius, role, gp, rec.origin, rec.dims, rec.spacing)
            ev[1].record(eng.stream)
            eng.dock(grid, ligs, *dock_args, seed=cfg.philox_seed, pose_stride=stride, out=out, chain_base=chain_base)
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
    pk = peaks()
    mc_ms = float(np.mean(t_mc))
    ach = w["flop"] / (mc_ms * 1e-3) / 1e12
    res = dict(
        workload=name, title=cfg.title, n_lig=L, n_chains=cfg.n_chains, n_steps=cfg.n_steps, top_k=k,
        evals=evals_all, value=evals_all / (ms * 1e-3), score_grad_evals_per_s=sg_all / (ms * 1e-3),
        ms_per_step=ms, ms_per_task=ms / max(batch_all.n_lig, 1) * (1 if scaling == "strong" else 1),
        ms_grid_build=float(np.mean(t_grid)), ms_mc_kernels=mc_ms, ms_topk=float(np.mean(t_topk)),
        wall_s=wall, launches=launches, scaling=scaling, clocks=clocks,
        roofline=dict(bound="alu", achieved=ach, peak=pk["alu_tflops"], unit="TFLOP/s", frac=ach / pk["alu_tflops"],
                      traffic=NCU_TRAFFIC_BYTES.get(name) if n_lig is None else None,
                      kernel=KERNEL_NAMES.get(eng.last_kernel(), "?") + ", fused MC step series",
                      peak_source=f"148 SM x 128 lanes x 2 x {pk['sm_mhz']:.0f} MHz ({pk['source']})",
                      xu_gops=w["xu"] / (mc_ms * 1e-3) / 1e9, xu_frac=w["xu"] / (mc_ms * 1e-3) / 1e9 / pk["xu_gops"],
                      grid_gather_gbs=w["gather_bytes"] / (mc_ms * 1e-3) / 1e9,
                      mc_kernel_evals_per_s=w["evals"] / (mc_ms * 1e-3)),
        best_energy=float(out[0][:, 0, 0].min().item()))
    if do_e2e:                                                               # host buffers in, host buffers out
        h_out = (np.empty((L, k, 2), np.float32), np.empty((L, k, stride), np.float32), np.empty((L, k), np.int32))
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
        h_xyz, h_typ = pin(rec.xyz), pin(rec.type)

        def e2e_step():
            lg = eng.load_ligands(batch, radius, role)
            grid = eng.build_grid(h_xyz, h_typ, radius, role, gp, rec.origin, rec.dims, rec.spacing)
            eng.dock(grid, lg, *dock_args, seed=cfg.philox_seed, pose_stride=stride, out=h_out, chain_base=chain_base)
            grid.free(); lg.free()
        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            e2e_step()
        barrier()
        e2e_s = (time.perf_counter() - t0) / steps
        if world > 1:
            tt = torch.tensor([e2e_s], device=eng.device)
            torch.distributed.all_reduce(tt, op=torch.distributed.ReduceOp.MAX)
            e2e_s = float(tt[0])
        h2d = rec.xyz.nbytes + rec.type.nbytes + sum(getattr(batch, f).nbytes for f in (
            "atom_off", "ref_xyz", "atom_type", "atom_frag", "tor_off", "tor_a", "tor_b", "tor_parent", "bond_off", "bond_ab"))
        res["e2e"] = dict(value=evals_all / e2e_s, unit=UNIT, h2d_bytes_per_step=int(h2d),
                          d2h_bytes_per_step=int(sum(a.nbytes for a in h_out)), ms_per_step=e2e_s * 1e3)
        assert np.array_equal(h_out[2], out[2].cpu().numpy()), "e2e and device-resident legs disagree"
    ligs.free()
    return res


# ----------------------------------------------------------------------------------------- oracle (CPU) arm
def oracle_setup(name, n_lig):
    from oracle import oracle as orc
    cfg = synth.CONFIGS[name]
    rec = synth.make_receptor(cfg)
    radius, role = synth.type_table(cfg.n_types)
    batch = synth.make_ligands(cfg, n_lig)
    p = orc.default_params()
    p.n_refine = cfg.n_refine
    return orc, cfg, rec, orc.Types(radius, role), p, batch


def oracle_time(name, budget_s=20.0, grid=None):
    """The oracle as it stands on the host cores: a0 in full (once), then a bounded sample of chains x steps."""
    cores = os.cpu_count() or 1
    orc, cfg, rec, ty, p, batch = oracle_setup(name, 1)
    t0 = time.perf_counter()
    G = grid or orc.build_grid(p, ty, rec.xyz, rec.type, rec.origin, rec.dims, rec.spacing)
    t_grid = time.perf_counter() - t0
    L = orc.ligand_from_batch(batch, 0)
    n_ch = min(cfg.n_chains, max(cores, 8) * 8)

    def dock(ns):
        t = time.perf_counter()
        orc.dock(p, ty, G, L, cfg.philox_seed, 0, n_ch, ns, rec.box_min, rec.box_max, rec.pocket_center, rec.pocket_radius)
        return time.perf_counter() - t
    t_probe = dock(4)
    ns = int(max(4, min(cfg.n_steps, 4 * budget_s / max(t_probe, 1e-6))))
    t_dock = dock(ns)
    evals_s = n_ch * (ns * (p.n_refine + 1) + 1)
    return dict(G=G, cores=cores, t_grid=t_grid, t_dock=t_dock, evals_sample=evals_s, dock_evals_per_s=evals_s / t_dock,
                sample=f"{name}: oracle grid build in full ({t_grid:.1f} s, OpenMP over nodes) + dock of ligand 0, "
                       f"{n_ch} chains x {ns} of {cfg.n_steps} steps ({t_dock:.1f} s)")


def cpu_baseline(name, w_evals_per_lig_step, n_lig_full, budget_s=20.0):
    """Whole-step oracle throughput estimate: full a0 time + sampled dock rate scaled to the step's evaluations."""
    r = oracle_time(name, budget_s)
    t_step = r["t_grid"] + w_evals_per_lig_step * n_lig_full / r["dock_evals_per_s"]
    return dict(value=w_evals_per_lig_step * n_lig_full / t_step, unit=UNIT, cores=r["cores"], kind="oracle",
                sample=r["sample"], dock_only_evals_per_s=r["dock_evals_per_s"], grid_build_s=r["t_grid"])


def run_reference(args):
    """--impl reference: the fp64 oracle on the host cores; each step = a bounded sample of the workload."""
    name = args.workload
    cfg = synth.CONFIGS[name]
    first = oracle_time(name, budget_s=8.0)
    vals = [first]
    for _ in range(max(args.warmup - 1, 0) + args.steps):
        vals.append(oracle_time(name, budget_s=8.0, grid=first["G"]))
    timed = vals[-args.steps:]
    rate = float(np.mean([v["dock_evals_per_s"] for v in timed]))
    evals_step = cfg.n_lig * cfg.n_chains * (cfg.n_steps * (cfg.n_refine + 1) + 1)
    t_step = first["t_grid"] + evals_step / rate
    value = evals_step / t_step
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=t_step * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=f"{name} {cfg.title} (BASELINE.json configs[{int(name[1]) - 1}])",
                            note="ms_per_step = measured full grid build + sampled dock rate scaled to the full step"),
                cpu_baseline=dict(value=value, unit=UNIT, kind="oracle", cores=first["cores"], sample=first["sample"]),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


# ----------------------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C2", choices=sorted(synth.CONFIGS))
    ap.add_argument("--impl", default="tridsk", choices=["tridsk", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the other configs' short runs")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle cpu_baseline leg")
    ap.add_argument("--n-lig", type=int, default=None, help="first n ligands of a screening config (profiling)")
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
    args.warmup = max(args.warmup, 3)
    main_res = run_workload(eng, args.workload, args.steps, args.warmup, rank, world, n_lig=args.n_lig)
    extras = {}
    if not args.no_extras and world == 1 and args.n_lig is None:
        for name in sorted(synth.CONFIGS):
            if name == args.workload:
                continue
            big = name in ("C3", "C5")
            r = run_workload(eng, name, 2 if big else 5, 3, do_e2e=False, sample_clocks=False)
            extras[name] = {k: r[k] for k in ("title", "evals", "value", "score_grad_evals_per_s", "ms_per_step", "ms_per_task",
                                              "ms_grid_build", "ms_mc_kernels", "ms_topk", "launches", "best_energy")}
            extras[name]["kernel"] = r["roofline"]["kernel"]
            extras[name]["roofline_frac"] = r["roofline"]["frac"]
            extras[name]["mc_kernel_evals_per_s"] = r["roofline"]["mc_kernel_evals_per_s"]
    if rank != 0:
        return
    cfg = synth.CONFIGS[args.workload]
    cpu = None
    if not args.no_cpu and args.n_lig is None:
        cpu = cpu_baseline(args.workload, cfg.n_chains * (cfg.n_steps * (cfg.n_refine + 1) + 1), cfg.n_lig)
    idx = int(args.workload[1]) - 1 if args.workload[0] == "C" else -1
    line = dict(
        metric=METRIC, value=main_res["value"], unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
        ms_per_step=main_res["ms_per_step"], higher_is_better=True, scaling=main_res["scaling"], vs_baseline=None,
        dtype="f32", data="synthetic",
        config=dict(workload=f"{args.workload} {cfg.title}" + (f" (BASELINE.json configs[{idx}])" if idx >= 0 else " (not a BASELINE.json config)"), n_ligands=main_res["n_lig"] * world
                    if main_res["scaling"] == "strong" else main_res["n_lig"], n_chains=cfg.n_chains, n_mc_steps=cfg.n_steps,
                    top_k=cfg.top_k, n_refine=cfg.n_refine, l2="flushed between steps (256 MiB memset outside the timed events)",
                    step="grid build (a0) + init + MC steps + top-k (a1..a10), one CUDA-graph launch"),
        score_grad_evals_per_s=main_res["score_grad_evals_per_s"], ms_per_task=main_res["ms_per_task"],
        ms_grid_build=main_res["ms_grid_build"], ms_mc_kernels=main_res["ms_mc_kernels"], ms_topk=main_res["ms_topk"],
        clocks=main_res["clocks"], e2e=main_res.get("e2e"), gpu_launches=main_res["launches"],
        roofline=main_res["roofline"], cpu_baseline=cpu, best_energy=main_res["best_energy"], other_workloads=extras)
    print(json.dumps(line))
    eng.close()
    if world > 1:
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
