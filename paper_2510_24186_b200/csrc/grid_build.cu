// grid_build.cu -- hot-path step a0: receptor grid precompute (O3/O4).
//
// G[t][k][j][i] = sum_a e(s_a, t, |x_node - r_a|).  One thread per grid node accumulates ALL ligand types in
// registers (the distance to a receptor atom is type-independent; only d_vdw and the donor/acceptor flag
// change), receptor atoms are staged through shared memory in chunks and read as warp broadcasts, and each
// type plane is written with unit-stride stores along x.  Receptor atoms are visited in input order, so the
// fp32 sums are reproducible.  The bound is the XU/FP32 pipes (one ex2 per node-atom-type triple), not memory.
#include <algorithm>

#include "internal.h"

#define GB_BX 32
#define GB_BY 4
#define GB_CHUNK 512

// pair_tab[s][t] = {d_vdw + mu, d_clash (2.6 for donor/acceptor pairs else d_vdw), hb flag, 1/d_clash}
template <int NT>
__global__ void __launch_bounds__(GB_BX * GB_BY) grid_build_kernel(const float4* __restrict__ rec, int n_rec,
                                                                   const float4* __restrict__ pair_tab, int n_types,
                                                                   const DParams P, const DGrid G, float dc_max,
                                                                   float* __restrict__ out) {
    __shared__ float4 s_atom[GB_CHUNK];
    __shared__ float4 s_tab[TRIDSK_MAX_TYPES * NT];
    const int tid = threadIdx.y * GB_BX + threadIdx.x;
    for (int i = tid; i < n_types * NT; i += GB_BX * GB_BY) {
        const int s = i / NT, t = i % NT;
        s_tab[i] = t < n_types ? pair_tab[s * n_types + t] : make_float4(0.f, 0.f, 0.f, 1.f);
    }
    const int ix = blockIdx.x * GB_BX + threadIdx.x, iy = blockIdx.y * GB_BY + threadIdx.y, iz = blockIdx.z;
    const bool in = ix < G.nx && iy < G.ny;
    const float x = G.ox + G.h * (float)ix, y = G.oy + G.h * (float)iy, z = G.oz + G.h * (float)iz;
    float acc[NT];
#pragma unroll
    for (int t = 0; t < NT; ++t) acc[t] = 0.f;
    const float dmax2 = P.long_dmax * P.long_dmax;

    for (int base = 0; base < n_rec; base += GB_CHUNK) {
        __syncthreads();
        for (int i = tid; i < GB_CHUNK && base + i < n_rec; i += GB_BX * GB_BY) s_atom[i] = rec[base + i];
        __syncthreads();
        const int cnt = min(GB_CHUNK, n_rec - base);
        for (int a = 0; a < cnt; ++a) {
            const float4 ra = s_atom[a];
            const float dx = x - ra.x, dy = y - ra.y, dz = z - ra.z;
            const float d2 = dx * dx + dy * dy + dz * dz;
            if (d2 >= dmax2) continue;
            const float rinv = rsqrtf(fmaxf(d2, 1e-12f));
            const float d = d2 * rinv;
            if (!(d < P.long_dmax)) continue;
            const float4* row = s_tab + __float_as_int(ra.w) * NT;
            if (d >= dc_max) {                      // common case: only the long-range Gaussian can act
#pragma unroll
                for (int t = 0; t < NT; ++t) {
                    const float u = d - row[t].x;
                    acc[t] -= P.w_long * __expf(-u * u * P.long_inv_two_sigma2);
                }
            } else {
                const float dfl = fmaxf(d, P.d_floor);
#pragma unroll
                for (int t = 0; t < NT; ++t) {
                    const float4 c = row[t];
                    const float u = d - c.x;
                    float e = -P.w_long * __expf(-u * u * P.long_inv_two_sigma2);
                    if (d < c.y) e -= P.w_clash * __logf(dfl * c.w);
                    if (c.z != 0.f && d < P.hb_dmax) {
                        const float w = d - P.hb_mu;
                        e -= P.w_hbond * __expf(-w * w * P.hb_inv_two_sigma2);
                    }
                    acc[t] += e;
                }
            }
        }
    }
    if (in) {
        const size_t node = ((size_t)iz * G.ny + iy) * G.nx + ix;
#pragma unroll
        for (int t = 0; t < NT; ++t)
            if (t < n_types) out[(size_t)t * G.plane + node] = acc[t];
    }
}

cudaError_t launch_grid_build(cudaStream_t s, const float4* rec, int n_rec, const float* pair_tab, int n_types,
                              const DParams& P, DGrid grid, float dc_max, float* out) {
    // dc_max >= every d_clash and hb_dmax: beyond it only the long-range Gaussian can act
    const dim3 block(GB_BX, GB_BY), g((grid.nx + GB_BX - 1) / GB_BX, (grid.ny + GB_BY - 1) / GB_BY, grid.nz);
    const float4* tab = reinterpret_cast<const float4*>(pair_tab);
    if (n_types <= 8) grid_build_kernel<8><<<g, block, 0, s>>>(rec, n_rec, tab, n_types, P, grid, dc_max, out);
    else if (n_types <= 16) grid_build_kernel<16><<<g, block, 0, s>>>(rec, n_rec, tab, n_types, P, grid, dc_max, out);
    else grid_build_kernel<32><<<g, block, 0, s>>>(rec, n_rec, tab, n_types, P, grid, dc_max, out);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ xy-packed copy of the grid (DGrid::gp)
// gp[t][z][y][x] = {g(x,y), g(x+1,y), g(x,y+1), g(x+1,y+1)} at the same (t, z); indices clamped at the upper
// edges (those records are never the base of a cell: i0 <= n - 2).  The 8 corners of a trilinear cell are then two
// aligned 16-byte records, which is what the chain kernels gather.
__global__ void __launch_bounds__(256) grid_pack_kernel(const DGrid G, float4* __restrict__ out) {
    const size_t total = G.plane * (size_t)G.n_types;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % G.nx), y = (int)((i / G.nx) % G.ny);
        const int dx = (x + 1 < G.nx) ? 1 : 0;
        const size_t dy = (y + 1 < G.ny) ? (size_t)G.nx : 0;
        out[i] = make_float4(G.g[i], G.g[i + dx], G.g[i + dy], G.g[i + dy + dx]);
    }
}

cudaError_t launch_grid_pack(cudaStream_t s, DGrid grid, float4* out) {
    const size_t total = grid.plane * (size_t)grid.n_types;
    const int blocks = (int)std::min<size_t>((total + 255) / 256, 148 * 16);
    grid_pack_kernel<<<blocks, 256, 0, s>>>(grid, out);
    return cudaGetLastError();
}
