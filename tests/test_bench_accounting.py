"""bench.py's accounting against the evaluation counts SURVEY.md 8(a) states for the BASELINE.json configs (no GPU)."""
import numpy as np

import bench
from workloads import synth

# "Evaluations (FK+score) per config, with n_refine = 1 -> 2 per MC step (+1 per chain at init)"
SURVEY_EVALS = {"C1": 12_864, "C2": 768_384, "C3": 524_812_288, "C4": 4_097_024, "C5": 2_520_776_704}


def test_evaluation_counts_match_the_survey():
    for name, want in SURVEY_EVALS.items():
        cfg = synth.CONFIGS[name]
        n = np.full(cfg.n_lig, 30)
        w = bench.work_of(n, np.full(cfg.n_lig, 5), np.full(cfg.n_lig, 300), cfg.n_chains, cfg.n_steps, cfg.n_refine)
        assert int(w["evals"]) == want, name
        assert int(w["sg_evals"]) == cfg.n_lig * cfg.n_chains * cfg.n_steps * cfg.n_refine      # the metric's strict count


def test_work_model_two_kinds_of_evaluation():
    """One chain, one step, n_refine = 1: one gradient evaluation + Adam, two energy evaluations (initial + Metropolis)."""
    N, T, P = 30, 6, 310
    w = bench.work_of([N], [T], [P], 1, 1, 1)
    g = 28 * P + 116 * N + 140 * T + 20 * (6 + T)
    e = 16 * P + 66 * N + 110 * T
    assert w["flop"] == g + 2 * e and w["gather_bytes"] == 3 * 32 * N
    # more refinement steps add gradient evaluations only
    w3 = bench.work_of([N], [T], [P], 1, 1, 3)
    assert w3["flop"] == 3 * g + 2 * e and w3["sg_evals"] == 3 and w3["evals"] == 5
    # the bound named is the one that needs the most time
    pk = dict(alu_tflops=1.0, xu_gops=1e9, sm_mhz=1965.0, source="test", l2_read_gbs=1e9)
    r = bench.roofline_of(w, 1.0, pk, "k")
    assert r["bound"] == "alu" and r["frac"] == r["alu_frac"] and abs(r["alu_frac"] - w["flop"] / 1e12 / 1e-3) < 1e-12
