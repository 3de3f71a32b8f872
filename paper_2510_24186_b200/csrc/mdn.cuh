// mdn.cuh -- the mixture-density term of the paper's score on the device (O15; Eq.GMM, Eq.E_MDN):
//   E_MDN = - sum_i sum_j [d_ij < d_cut] sum_k pi_ijk N(d_ij; mu_ijk, sigma_ijk),   d_ij = min over the atoms of residue i
// of the distance to ligand atom j, N the normalised Gaussian density (G17); the gradient flows through the arg-min
// atom, ties of the minimum go to the lowest atom index, indicators are not differentiated (G21).
// It is a per-ligand-atom term like the grid lookup (it sees only x_j), so every mapping of the fused kernel calls
// mdn_atom() at the place where it interpolates the receptor grid for an atom.  This is the paper's own "self-defined
// kernel function" that skips far pairs (P:353 item 4): a residue is visited only if the cell list (internal.h) names
// it for the cell the atom is in.
#pragma once
#include "internal.h"

// One ligand atom (internal index p of a ligand with n atoms) at (x, y, z) against residues i0, i0 + istep, ...
// par = the ligand's parameter block [n_res][n][K] of {a, mu, nk2, 1/sigma^2}, a = w_mdn pi / (sigma sqrt(2 pi)),
// nk2 = -log2(e) / (2 sigma^2):  N = a 2^(nk2 (d - mu)^2),  dN/dd = -N (d - mu) / sigma^2.
// e += w_mdn * (this atom's share of E_MDN); grad: (gx, gy, gz) += its gradient.
// two adjacent 16-byte records by one 256-bit load (p 32-byte aligned)
__device__ __forceinline__ void mdn_ldg2(const float4* p, float4& a, float4& b) {
    asm("ld.global.nc.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
        : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w) : "l"(p));
}

// One (residue, atom) pair whose minimum squared distance best2 is inside the cut-off: the K mixture components.  The
// records are padded to a multiple of four per pair (M.K4; the padding has zero amplitude) and fetched four at a time by two
// 256-bit loads; the first four (c0) were requested by the caller before it searched the residue's atoms.
__device__ __forceinline__ void mdn_finish(const MdnDev& M, const float4* __restrict__ q, const float4 c0[8], float best2,
                                           float bx, float by, float bz, bool grad, float& e, float& gx, float& gy, float& gz) {
    float rinv;
    { const float b = fmaxf(best2, 1e-12f); asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(b)); }
    const float d = best2 * rinv;
    float de = 0.f;
    float4 c[4] = {c0[0], c0[1], c0[2], c0[3]};
    for (int k0 = 0; k0 < M.K4; k0 += 4) {
        float4 cn[4];
        const bool more = k0 + 4 < M.K4;
        if (more) {
            if (k0 == 0) { cn[0] = c0[4]; cn[1] = c0[5]; cn[2] = c0[6]; cn[3] = c0[7]; }      // the second four came with the first
            else { mdn_ldg2(q + k0 + 4, cn[0], cn[1]); mdn_ldg2(q + k0 + 6, cn[2], cn[3]); }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float t = d - c[j].y;
            float N;
            { const float arg = c[j].z * t * t; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(N) : "f"(arg)); }
            N *= c[j].x;
            e -= N;
            de = fmaf(N * t, c[j].w, de);
        }
        if (more) {
#pragma unroll
            for (int j = 0; j < 4; ++j) c[j] = cn[j];
        }
    }
    if (grad) {
        const float sc = de * rinv;
        gx = fmaf(sc, bx, gx); gy = fmaf(sc, by, gy); gz = fmaf(sc, bz, gz);
    }
}

__device__ __forceinline__ void mdn_atom(const MdnDev& M, const float4* __restrict__ par, int n, int p, float x, float y, float z,
                                         int i0, int istep, bool grad, float& e, float& gx, float& gy, float& gz) {
    // the cell of the atom streams every receptor atom it can be within d_cut of, sorted by residue (outside the grid: none)
    const float ux = (x - M.glo[0]) * M.inv_cell, uy = (y - M.glo[1]) * M.inv_cell, uz = (z - M.glo[2]) * M.inv_cell;
    const int ix = __float2int_rd(ux), iy = __float2int_rd(uy), iz = __float2int_rd(uz);
    if ((unsigned)ix >= (unsigned)M.nc[0] || (unsigned)iy >= (unsigned)M.nc[1] || (unsigned)iz >= (unsigned)M.nc[2]) return;
    const int cell = (iz * M.nc[1] + iy) * M.nc[0] + ix;
    const int e0 = __ldg(M.cell_off + cell), e1 = __ldg(M.cell_off + cell + 1);
    if (e0 >= e1) return;
    const float cut2 = M.d_cut * M.d_cut;
    // Residue by residue: the first entry of a run holds residue id | run length << 16; runs are padded to an even number of
    // entries (a padding entry lies 1e18 away) so that every run starts 32-byte aligned and is read two entries per 256-bit
    // load.  Lanes of a warp sit in different cells, so their runs differ in length; the short inner loop diverges, the costly
    // mixture evaluation after it is reached by all lanes together once per residue.  The loads are L2 round trips: the first
    // four parameter records of the residue and the first entries of the NEXT run are requested before the run is searched.
    int ord = 0;
    float4 a, a2;
    mdn_ldg2(M.cell_at + e0, a, a2);
    for (int en = e0; en < e1; ++ord) {
        const int hdr = __float_as_int(a.w), i = hdr & 0xffff, cnt = hdr >> 16;      // cnt is even
        const float4* q = par + ((size_t)i * n + p) * M.K4;
        float4 c0[8];                                         // K4 >= 8 ? eight records : four (the rest of c0 is unused then)
        mdn_ldg2(q, c0[0], c0[1]); mdn_ldg2(q + 2, c0[2], c0[3]);
        if (M.K4 > 4) { mdn_ldg2(q + 4, c0[4], c0[5]); mdn_ldg2(q + 6, c0[6], c0[7]); }
        float4 an, an2;
        mdn_ldg2(M.cell_at + min(en + cnt, e1 - 2), an, an2);
        float bx = x - a.x, by = y - a.y, bz = z - a.z;
        float best2 = bx * bx + by * by + bz * bz;
        {
            const float dx = x - a2.x, dy = y - a2.y, dz = z - a2.z;
            const float d2 = dx * dx + dy * dy + dz * dz;
            if (d2 < best2) { best2 = d2; bx = dx; by = dy; bz = dz; }
        }
        for (int r = 2; r < cnt; r += 2) {                    // plain minimum, ties -> lowest atom index
            float4 b0, b1;
            mdn_ldg2(M.cell_at + en + r, b0, b1);
            float dx = x - b0.x, dy = y - b0.y, dz = z - b0.z;
            float d2 = dx * dx + dy * dy + dz * dz;
            if (d2 < best2) { best2 = d2; bx = dx; by = dy; bz = dz; }
            dx = x - b1.x; dy = y - b1.y; dz = z - b1.z;
            d2 = dx * dx + dy * dy + dz * dz;
            if (d2 < best2) { best2 = d2; bx = dx; by = dy; bz = dz; }
        }
        en += cnt;
        if (best2 < cut2 && ord % istep == i0) mdn_finish(M, q, c0, best2, bx, by, bz, grad, e, gx, gy, gz);
        a = an; a2 = an2;
    }
}
