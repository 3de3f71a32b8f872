// mdn.cuh -- the mixture-density term of the paper's score on the device (O15; Eq.GMM, Eq.E_MDN):
//   E_MDN = - sum_i sum_j [d_ij < d_cut] sum_k pi_ijk N(d_ij; mu_ijk, sigma_ijk),   d_ij = min over the atoms of residue i
// of the distance to ligand atom j, N the normalised Gaussian density (G17); the gradient flows through the arg-min
// atom, ties of the minimum go to the lowest atom index, indicators are not differentiated (G21).
// It is a per-ligand-atom term like the grid lookup (it sees only x_j), so every mapping of the fused kernel calls
// mdn_atom() at the place where it interpolates the receptor grid for an atom.  This is the paper's own "self-defined
// kernel function" that skips far pairs (P:353 item 4): a residue is visited only if the atom lies inside its bounding
// sphere grown by d_cut.
#pragma once
#include "internal.h"

// One ligand atom (internal index p of a ligand with n atoms) at (x, y, z) against residues i0, i0 + istep, ...
// par = the ligand's parameter block [n_res][n][K] of {a, mu, nk2, 1/sigma^2}, a = w_mdn pi / (sigma sqrt(2 pi)),
// nk2 = -log2(e) / (2 sigma^2):  N = a 2^(nk2 (d - mu)^2),  dN/dd = -N (d - mu) / sigma^2.
// e += w_mdn * (this atom's share of E_MDN); grad: (gx, gy, gz) += its gradient.
__device__ __forceinline__ void mdn_atom(const MdnDev& M, const float4* __restrict__ par, int n, int p, float x, float y, float z,
                                         int i0, int istep, bool grad, float& e, float& gx, float& gy, float& gz) {
    for (int i = i0; i < M.n_res; i += istep) {
        const float4 s = __ldg(M.sph + i);                    // centre, (bounding radius + d_cut)^2
        const float sx = x - s.x, sy = y - s.y, sz = z - s.z;
        if (!(sx * sx + sy * sy + sz * sz < s.w)) continue;
        float best2 = 3.0e38f, bx = 0.f, by = 0.f, bz = 0.f;
        const int r1 = __ldg(M.res_off + i + 1);
        for (int r = __ldg(M.res_off + i); r < r1; ++r) {     // plain minimum, ties -> lowest index
            const float4 a = __ldg(M.rec + r);
            const float dx = x - a.x, dy = y - a.y, dz = z - a.z;
            const float d2 = dx * dx + dy * dy + dz * dz;
            if (d2 < best2) { best2 = d2; bx = dx; by = dy; bz = dz; }
        }
        const float d = sqrtf(best2);
        if (!(d < M.d_cut)) continue;
        const float4* q = par + ((size_t)i * n + p) * M.K;
        float de = 0.f;
        for (int k = 0; k < M.K; ++k) {
            const float4 c = __ldg(q + k);
            const float t = d - c.y;
            float N;
            { const float arg = c.z * t * t; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(N) : "f"(arg)); }
            N *= c.x;
            e -= N;
            de = fmaf(N * t, c.w, de);
        }
        if (grad && d > 0.f) {
            const float sc = de / d;
            gx = fmaf(sc, bx, gx); gy = fmaf(sc, by, gy); gz = fmaf(sc, bz, gz);
        }
    }
}
