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

// Parameter layout (internal.h, mdn_slot_f4): a (residue, atom) pair owns one SLOT of blocks; a block holds up to ten
// components as {a, mu, nk2} x 10 (30 floats + 2 unused = 128 bytes, one cache line), a = w_mdn pi / (sigma sqrt(2 pi)),
// nk2 = -log2(e) / (2 sigma^2):  N = a 2^(nk2 (d - mu)^2),  dN/dd = -N (d - mu) / sigma^2 = 2 ln 2 N (d - mu) nk2.
// The last block is cut to whole 32-byte chunks; unused components have zero amplitude.  K <= 10 (the paper's mixture
// sizes): one block, fetched whole by the caller one residue AHEAD of its use.
__device__ __forceinline__ void mdn_ldg2(const float4* p, float4& a, float4& b) {     // two adjacent 16-byte records, p 32-byte aligned
    asm("ld.global.nc.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
        : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w) : "l"(p));
}
__device__ __forceinline__ void mdn_ldg8(const float4* p, float* v) {                  // one 32-byte chunk
    asm("ld.global.nc.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
        : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]) : "l"(p));
}
// the first nch (1..4, warp-uniform) chunks of the block at q
__device__ __forceinline__ void mdn_load_block(const float4* q, int nch, float v[32]) {
    mdn_ldg8(q, v);
    if (nch > 1) mdn_ldg8(q + 2, v + 8);
    if (nch > 2) mdn_ldg8(q + 4, v + 16);
    if (nch > 3) mdn_ldg8(q + 6, v + 24);
}
// the components that lie wholly inside the first nch chunks of a block: e -= sum N, dn += sum N (d - mu) nk2
__device__ __forceinline__ void mdn_block(const float v[32], int nch, float d, float& e, float& dn) {
#pragma unroll
    for (int j = 0; j < 10; ++j) {
        if (3 * j + 2 < 8 * nch) {
            const float t = d - v[3 * j + 1];
            float N;
            { const float arg = v[3 * j + 2] * t * t; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(N) : "f"(arg)); }
            N *= v[3 * j];
            e -= N;
            dn = fmaf(N * t, v[3 * j + 2], dn);
        }
    }
}

// One (residue, atom) pair whose minimum squared distance best2 is inside the cut-off: the K mixture components.  c0 = the
// slot's first block (requested by the caller one residue ahead); further blocks (K > 10) are fetched here.
__device__ __forceinline__ void mdn_finish(const MdnDev& M, const float4* __restrict__ q, const float c0[32], float best2,
                                           float bx, float by, float bz, bool grad, float& e, float& gx, float& gy, float& gz) {
    float rinv;
    { const float b = fmaxf(best2, 1e-12f); asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(b)); }
    const float d = best2 * rinv;
    float dn = 0.f;
    const int nch0 = min(M.K4 >> 1, 4);
    mdn_block(c0, nch0, d, e, dn);
    for (int c = 4; 2 * c < M.K4; c += 4) {                     // K > 10
        float v[32];
        const int nch = min((M.K4 >> 1) - c, 4);
        mdn_load_block(q + 2 * c, nch, v);
        mdn_block(v, nch, d, e, dn);
    }
    if (grad) {
        const float sc = -1.3862943611198906f * dn * rinv;      // de/dd / d,  1 / sigma^2 = -2 ln 2 nk2
        gx = fmaf(sc, bx, gx); gy = fmaf(sc, by, gy); gz = fmaf(sc, bz, gz);
    }
}

// One ligand atom (internal index p of a ligand with n atoms) at (x, y, z) against residues i0, i0 + istep, ...
// par = the ligand's parameter block [n_res][n] of slots (M.K4 float4 each).
// e += w_mdn * (this atom's share of E_MDN); grad: (gx, gy, gz) += its gradient.
// PIPE = false: the parameter block is requested only once its run has passed the cut-off test, by the lane that evaluates it
// (one buffer, no speculative loads: for the instances whose register budget cannot hold two).
template <bool PIPE = true>
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
    const int nch0 = min(M.K4 >> 1, 4);
    // Residue by residue.  The FIRST entry of a run holds residue id | run length << 16 in w, the SECOND the same header of the
    // NEXT run of the cell (-1: none); runs are padded to an even number of entries (a padding entry lies 1e18 away), so every
    // run starts 32-byte aligned and is read two entries per 256-bit load.  Everything a run needs -- its entries and the first
    // parameter block of its residue -- is requested while the run BEFORE it is being worked on: the loop is a one-ahead
    // software pipeline over L2 round trips.  Lanes of a warp sit in different cells, so their runs differ in length; the short
    // inner loop diverges, the costly mixture evaluation after it is reached by all lanes together once per residue.
    // The loop body is written once and instantiated twice with the two buffer sets swapped, so that no register copy touches
    // a load that is still in flight.
    int ord = 0, en = e0;
    float4 a, a2, b, b2;
    float cur[32], nxt[32];
    mdn_ldg2(M.cell_at + e0, a, a2);
    int hdr = __float_as_int(a.w);
    if (PIPE) mdn_load_block(par + ((size_t)(hdr & 0xffff) * n + p) * M.K4, nch0, cur);
    auto step = [&](const float4& ra, const float4& ra2, const float (&rc)[32], float4& na, float4& na2, float (&nc)[32]) {
        const int i = hdr & 0xffff, cnt = hdr >> 16;             // cnt is even
        const float4* q = par + ((size_t)i * n + p) * M.K4;
        const int nh = __float_as_int(ra2.w);                    // the next run's header
        if (nh >= 0) {
            mdn_ldg2(M.cell_at + en + cnt, na, na2);
            if (PIPE) mdn_load_block(par + ((size_t)(nh & 0xffff) * n + p) * M.K4, nch0, nc);
        }
        float bx = x - ra.x, by = y - ra.y, bz = z - ra.z;
        float best2 = bx * bx + by * by + bz * bz;
        {
            const float dx = x - ra2.x, dy = y - ra2.y, dz = z - ra2.z;
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
        if (best2 < cut2 && ord % istep == i0) {
            if (!PIPE) mdn_load_block(q, nch0, nc);             // (nc and rc are the same buffer then)
            mdn_finish(M, q, rc, best2, bx, by, bz, grad, e, gx, gy, gz);
        }
        en += cnt; hdr = nh; ++ord;
    };
    for (;;) {
        step(a, a2, cur, b, b2, PIPE ? nxt : cur);
        if (en >= e1) break;
        step(b, b2, PIPE ? nxt : cur, a, a2, cur);
        if (en >= e1) break;
    }
}

// The same term for the mapping whose lanes SHARE an atom (CTA per chain, pair-record instance): lane i0 of the atom's istep
// lanes takes the candidate runs i0, i0 + istep, ... of the cell through the run directory (internal.h) instead of walking
// the whole stream -- the same assignment as mdn_atom's `ord % istep == i0`, so every lane's partial sum is the same, in a
// quarter (an eighth, a half) of the dependent L2 round trips.  One buffer: the parameter block is requested once the run has
// passed the cut-off test; the directory entry of the lane's next run is requested one run ahead.
__device__ __forceinline__ void mdn_atom_shared(const MdnDev& M, const float4* __restrict__ par, int n, int p, float x, float y, float z,
                                                int i0, int istep, bool grad, float& e, float& gx, float& gy, float& gz) {
    const float ux = (x - M.glo[0]) * M.inv_cell, uy = (y - M.glo[1]) * M.inv_cell, uz = (z - M.glo[2]) * M.inv_cell;
    const int ix = __float2int_rd(ux), iy = __float2int_rd(uy), iz = __float2int_rd(uz);
    if ((unsigned)ix >= (unsigned)M.nc[0] || (unsigned)iy >= (unsigned)M.nc[1] || (unsigned)iz >= (unsigned)M.nc[2]) return;
    const int cell = (iz * M.nc[1] + iy) * M.nc[0] + ix;
    const int d1 = __ldg(M.dir_off + cell + 1);
    int k = __ldg(M.dir_off + cell) + i0;
    if (k >= d1) return;
    const float cut2 = M.d_cut * M.d_cut;
    const int nch0 = min(M.K4 >> 1, 4);
    int2 de = __ldg(M.dir + k);
    for (; k < d1; k += istep) {
        const int hdr = de.x, en = de.y, cnt = hdr >> 16;         // cnt is even
        float4 a, a2;
        mdn_ldg2(M.cell_at + en, a, a2);
        const int2 dn = __ldg(M.dir + min(k + istep, d1 - 1));    // this lane's next run (or a harmless re-read)
        float bx = x - a.x, by = y - a.y, bz = z - a.z;
        float best2 = bx * bx + by * by + bz * bz;
        {
            const float dx = x - a2.x, dy = y - a2.y, dz = z - a2.z;
            const float d2 = dx * dx + dy * dy + dz * dz;
            if (d2 < best2) { best2 = d2; bx = dx; by = dy; bz = dz; }
        }
        for (int r = 2; r < cnt; r += 2) {                        // plain minimum, ties -> lowest atom index
            float4 b0, b1;
            mdn_ldg2(M.cell_at + en + r, b0, b1);
            float dx = x - b0.x, dy = y - b0.y, dz = z - b0.z;
            float d2 = dx * dx + dy * dy + dz * dz;
            if (d2 < best2) { best2 = d2; bx = dx; by = dy; bz = dz; }
            dx = x - b1.x; dy = y - b1.y; dz = z - b1.z;
            d2 = dx * dx + dy * dy + dz * dz;
            if (d2 < best2) { best2 = d2; bx = dx; by = dy; bz = dz; }
        }
        if (best2 < cut2) {
            const float4* q = par + ((size_t)(hdr & 0xffff) * n + p) * M.K4;
            float v[32];
            mdn_load_block(q, nch0, v);
            mdn_finish(M, q, v, best2, bx, by, bz, grad, e, gx, gy, gz);
        }
        de = dn;
    }
}
