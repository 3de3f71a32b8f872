"""oracle/mdn.py -- E_MDN, the mixture-density term of the paper's score, as a plain fp64 definition.

TEST INFRASTRUCTURE (like the rest of oracle/): only tests/ may import it; it shares no code with the CUDA path.
STATUS: the plain Python transcription of O15.  The oracle the kernels are checked against is orc_mdn_energy in
tridsk_oracle.c (the same definition in C, called from orc_score_grad / orc_mc_step); both run under the same pins in
tests/test_oracle_pins.py and must agree with each other to rounding.

What is computed (P:N = /root/reference/PAPER.md line N):
  Eq.GMM      p(d | i, j) = sum_k pi_ijk N(d; mu_ijk, sigma_ijk)      K Gaussians per (residue i, ligand atom j)
  Eq.E_MDN E_MDN = - sum_i sum_j [d_ij < d_cut] sum_k pi_ijk N(d_ij; mu_ijk, sigma_ijk),   d_cut = 5 A
  d_ij          the minimum distance between the atoms of residue i and ligand atom j
Readings: G1 the Gaussian exponent is negative (printed positive); G17 N is the NORMALISED density
exp(-(d-mu)^2 / (2 sigma^2)) / (sigma sqrt(2 pi)) (the prefactor is not printed) and K is the caller's (the paper does not
give it); G21 ties of the minimum go to the lowest receptor-atom index, and neither the arg-min switch nor the cut-off
indicator is differentiated (the gradient flows through the arg-min atom, as SURVEY 8(f) states).
"""
from __future__ import annotations

import math

import numpy as np


def mdn_energy(rec_xyz, res_off, pi, mu, sigma, x, d_cut=5.0):
    """rec_xyz[n_rec][3]; res_off[n_res+1] (the atoms of residue i are rec_xyz[res_off[i]:res_off[i+1]]);
    pi, mu, sigma [n_res][n][K]; x[n][3] ligand atom coordinates.
    -> (E_MDN, dE/dx [n][3], d [n_res][n] the minimum distances)."""
    rec_xyz = np.asarray(rec_xyz, dtype=np.float64)
    x = np.asarray(x, dtype=np.float64)
    pi, mu, sigma = (np.asarray(a, dtype=np.float64) for a in (pi, mu, sigma))
    n_res, n, K = pi.shape
    assert len(res_off) == n_res + 1 and x.shape == (n, 3)
    E = 0.0
    g = np.zeros((n, 3))
    dmin = np.zeros((n_res, n))
    for i in range(n_res):
        atoms = rec_xyz[res_off[i]:res_off[i + 1]]
        for j in range(n):
            best, r_best = math.inf, -1
            for r in range(len(atoms)):                      # plain minimum, ties -> lowest index (G21)
                d = math.sqrt(float(np.sum((x[j] - atoms[r]) ** 2)))
                if d < best:
                    best, r_best = d, r
            dmin[i, j] = best
            if not best < d_cut:                             # [d_ij < d_cut]
                continue
            dE_dd = 0.0
            for k in range(K):
                s, m, w = sigma[i, j, k], mu[i, j, k], pi[i, j, k]
                N = math.exp(-(best - m) ** 2 / (2.0 * s * s)) / (s * math.sqrt(2.0 * math.pi))
                E -= w * N
                dE_dd -= w * N * (-(best - m) / (s * s))
            if best > 0.0:
                g[j] += dE_dd * (x[j] - atoms[r_best]) / best
    return E, g, dmin
