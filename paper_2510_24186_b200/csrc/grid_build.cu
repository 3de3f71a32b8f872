// grid_build.cu -- hot-path step a0: receptor grid precompute (O3/O4).
//
// G[t][k][j][i] = sum_a e(s_a, t, |x_node - r_a|).  One thread per grid node accumulates ALL ligand types in
// registers (the distance to a receptor atom is type-independent; only d_vdw and the donor/acceptor flag change).
// A CTA owns a compact brick of 8 x 4 x 4 nodes (a warp: 8 x 2 x 2), so that the atoms within the 10 A cut-off of
// one lane are nearly those of the whole warp.  Receptor atoms stream through in chunks: the CTA first culls a chunk
// against the brick's bounding sphere (ordered compaction, so atoms are still visited in input order and the fp32
// sums are reproducible), then every thread walks the survivors as warp broadcasts from shared memory.
// The bound is the XU pipe (one ex2 per node-atom-type triple), not memory: the grid is written once.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "internal.h"

#define GB_BX 8
#define GB_BY 4
#define GB_BZ 4
#define GB_THREADS (GB_BX * GB_BY * GB_BZ)
#define GB_CHUNK 1024

__device__ __forceinline__ float exp2f_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// {x, y, z, type bits} per receptor atom; *bad is set if a type is out of range (the atom is then skipped)
__global__ void rec_pack_kernel(const float* __restrict__ xyz, const int* __restrict__ type, int n_rec, int n_types,
                                float4* __restrict__ out, int* __restrict__ bad) {
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n_rec) return;
    int t = type[a];
    if (t < 0 || t >= n_types) { *bad = 1; t = -1; }
    out[a] = make_float4(xyz[3 * a], xyz[3 * a + 1], xyz[3 * a + 2], __int_as_float(t));
}

// pair_tab[s][t] = {d_vdw + mu, d_clash (2.6 for donor/acceptor pairs else d_vdw), hb flag, 1/d_clash}
// LAT: the ligand types' radii lie on a lattice r_min + m delta with consecutive m (GridLattice, api.cu).  Then
// 2^(nk2 (x - m delta)^2) = A B^m C_m with x = d - r_s - mu - r_min, A = 2^(nk2 x^2), B = 2^(-2 nk2 delta x) and the
// constants C_m = 2^(nk2 m^2 delta^2): two ex2 per (node, atom) instead of one per type, the rest are multiplications --
// the kernel leaves the XU bound (1.08 -> 0.5 ms on C2).
struct GridLattice {
    int on;                       // 0: general table
    float delta_k;                // -2 nk2 delta
    float rmin;                   // smallest ligand-type radius
    unsigned step_mask;           // bit k: sorted type k has m one larger than sorted type k - 1 (else the same m)
    unsigned char order[TRIDSK_MAX_TYPES];   // sorted position k -> type
    float cm[TRIDSK_MAX_TYPES];   // C_m of sorted position k
};

// LAT: 0 general table, 1 lattice, 2 lattice whose sorted types all step up by one delta (no select per type)
template <int NT, int LAT>
__global__ void __launch_bounds__(GB_THREADS) grid_build_kernel(const float4* __restrict__ rec, int n_rec,
                                                                const float4* __restrict__ pair_tab, int n_types,
                                                                const DParams P, const DGrid G, float dc_max,
                                                                const GridLattice lat, const float* __restrict__ rec_radius,
                                                                float* __restrict__ out) {
    __shared__ float4 s_atom[GB_CHUNK];
    __shared__ float4 s_tab[TRIDSK_MAX_TYPES * NT];
    __shared__ __align__(16) float s_c[TRIDSK_MAX_TYPES * NT];      // d_vdw + mu alone: what the common case reads
    __shared__ int s_warp[GB_THREADS / 32 + 1];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < n_types * NT; i += GB_THREADS) {
        const int s = i / NT, t = i % NT;
        const float4 e = t < n_types ? pair_tab[s * n_types + t] : make_float4(1e15f, 0.f, 0.f, 1.f);
        s_tab[i] = e; s_c[i] = e.x;
    }
    // node of this thread: warp = 8 x 2 x 2 sub-brick, the CTA's 4 warps tile 8 x 4 x 4
    const int lx = lane & 7, ly = ((lane >> 3) & 1) + 2 * (warp & 1), lz = (lane >> 4) + 2 * (warp >> 1);
    const int ix = blockIdx.x * GB_BX + lx, iy = blockIdx.y * GB_BY + ly, iz = blockIdx.z * GB_BZ + lz;
    const bool in = ix < G.nx && iy < G.ny && iz < G.nz;
    const float x = G.ox + G.h * (float)ix, y = G.oy + G.h * (float)iy, z = G.oz + G.h * (float)iz;
    // bounding sphere of the brick
    const float hx = 0.5f * G.h * (float)(GB_BX - 1), hy = 0.5f * G.h * (float)(GB_BY - 1), hz = 0.5f * G.h * (float)(GB_BZ - 1);
    const float cx = G.ox + G.h * (float)(blockIdx.x * GB_BX) + hx, cy = G.oy + G.h * (float)(blockIdx.y * GB_BY) + hy;
    const float cz = G.oz + G.h * (float)(blockIdx.z * GB_BZ) + hz;
    // the indicators of O2 are independent: cull with the larger of the long-range cut-off and the clash / hydrogen-bond range
    const float cull = fmaxf(P.long_dmax, dc_max);
    const float rc = cull + sqrtf(hx * hx + hy * hy + hz * hz) + 1e-3f;
    const float rc2 = rc * rc;

    float acc[NT], accx[NT];                       // acc: sum of 2^(...) Gaussians (scaled by -w_long at the end); accx: the rest
#pragma unroll
    for (int t = 0; t < NT; ++t) { acc[t] = 0.f; accx[t] = 0.f; }
    const float dmax2 = cull * cull;
    const float nk2 = -P.long_inv_two_sigma2 * 1.4426950408889634f;

    for (int base = 0; base < n_rec; base += GB_CHUNK) {
        // ---- cull this chunk against the brick's sphere, keeping input order
        __syncthreads();
        int n_keep = 0;
        for (int r0 = 0; r0 < GB_CHUNK && base + r0 < n_rec; r0 += GB_THREADS) {
            const int a = base + r0 + tid;
            float4 ra = make_float4(0.f, 0.f, 0.f, 0.f);
            bool keep = false;
            if (a < n_rec) {
                ra = __ldg(rec + a);
                const float dx = ra.x - cx, dy = ra.y - cy, dz = ra.z - cz;
                keep = (dx * dx + dy * dy + dz * dz < rc2) && (__float_as_int(ra.w) >= 0);
            }
            const unsigned m = __ballot_sync(0xffffffffu, keep);
            if (lane == 0) s_warp[warp] = __popc(m);
            __syncthreads();
            int off = n_keep, total = 0;
#pragma unroll
            for (int w = 0; w < GB_THREADS / 32; ++w) { const int c = s_warp[w]; if (w < warp) off += c; total += c; }
            if (keep) s_atom[off + __popc(m & ((1u << lane) - 1u))] = ra;
            n_keep += total;
            __syncthreads();
        }
        // ---- every node against the survivors
        for (int a = 0; a < n_keep; ++a) {
            const float4 ra = s_atom[a];
            const float dx = x - ra.x, dy = y - ra.y, dz = z - ra.z;
            const float d2 = dx * dx + dy * dy + dz * dz;
            if (d2 >= dmax2) continue;
            const float rinv = rsqrtf(fmaxf(d2, 1e-12f));
            const float d = d2 * rinv;
            const int s = __float_as_int(ra.w);
            if (!(d < P.long_dmax)) {               // beyond the long-range cut-off: only the rare terms below can act
                if (!(d < dc_max)) continue;
            } else if (LAT) {
                const float xs = d - s_c[s * NT + lat.order[0]];      // r_s + r_min + mu, as tabulated
                const float B = exp2f_approx(lat.delta_k * xs);
                float pw = exp2f_approx(nk2 * xs * xs);
#pragma unroll
                for (int k = 0; k < NT; ++k) {                  // sorted by radius; padding positions have cm = 0
                    if (k > 0) pw = (LAT == 2 || ((lat.step_mask >> k) & 1u)) ? pw * B : pw;
                    acc[k] = fmaf(pw, lat.cm[k], acc[k]);
                }
            } else {
            const float4* crow = reinterpret_cast<const float4*>(s_c + s * NT);
#pragma unroll
            for (int t4 = 0; t4 < NT / 4; ++t4) {
                const float4 c = crow[t4];
                const float u0 = d - c.x, u1 = d - c.y, u2 = d - c.z, u3 = d - c.w;
                acc[4 * t4 + 0] += exp2f_approx(u0 * (u0 * nk2));
                acc[4 * t4 + 1] += exp2f_approx(u1 * (u1 * nk2));
                acc[4 * t4 + 2] += exp2f_approx(u2 * (u2 * nk2));
                acc[4 * t4 + 3] += exp2f_approx(u3 * (u3 * nk2));
            }
            }
            if (d < dc_max) {                       // rare: clash and / or hydrogen-bond range of some type
                const float4* row = s_tab + s * NT;
                const float dfl = fmaxf(d, P.d_floor);
#pragma unroll
                for (int t = 0; t < NT; ++t) {
                    const float4 c = row[t];
                    float e = 0.f;
                    if (d < c.y) e -= P.w_clash * __logf(dfl * c.w);
                    if (c.z != 0.f && d < P.hb_dmax) {
                        const float w = d - P.hb_mu;
                        e -= P.w_hbond * __expf(-w * w * P.hb_inv_two_sigma2);
                    }
                    accx[t] += e;
                }
            }
        }
    }
    if (in) {
        const size_t node = ((size_t)iz * G.ny + iy) * G.nx + ix;
        if (LAT) {                                              // acc is in sorted order, accx in type order
#pragma unroll
            for (int k = 0; k < NT; ++k)
                if (k < n_types) { const int t = lat.order[k]; out[(size_t)t * G.plane + node] = -P.w_long * acc[k]; }
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if (t < n_types && accx[t] != 0.f) out[(size_t)t * G.plane + node] += accx[t];
        } else {
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if (t < n_types) out[(size_t)t * G.plane + node] = fmaf(-P.w_long, acc[t], accx[t]);
        }
    }
}

cudaError_t launch_rec_pack(cudaStream_t s, const float* xyz, const int* type, int n_rec, int n_types, float4* out, int* bad) {
    if (n_rec <= 0) return cudaSuccess;
    rec_pack_kernel<<<(n_rec + 255) / 256, 256, 0, s>>>(xyz, type, n_rec, n_types, out, bad);
    return cudaGetLastError();
}

cudaError_t launch_grid_build(cudaStream_t s, const float4* rec, int n_rec, const float* pair_tab, int n_types,
                              const DParams& P, DGrid grid, float dc_max, const float* radius_h, const float* rec_radius_dev,
                              float* out) {
    // dc_max >= every d_clash and hb_dmax: beyond it only the long-range Gaussian can act
    const dim3 g((grid.nx + GB_BX - 1) / GB_BX, (grid.ny + GB_BY - 1) / GB_BY, (grid.nz + GB_BZ - 1) / GB_BZ);
    const float4* tab = reinterpret_cast<const float4*>(pair_tab);
    // lattice detection (layout of the type table, no arithmetic of the method): sort the types by radius; the steps
    // between consecutive distinct radii must all equal one delta
    GridLattice lat;
    memset(&lat, 0, sizeof(lat));
    {
        int ord[TRIDSK_MAX_TYPES];
        for (int t = 0; t < n_types; ++t) ord[t] = t;
        std::stable_sort(ord, ord + n_types, [&](int x, int y) { return radius_h[x] < radius_h[y]; });
        double delta = 0.0;
        for (int k = 1; k < n_types; ++k) {
            const double df = (double)radius_h[ord[k]] - radius_h[ord[k - 1]];
            if (df > 1e-6 && (delta == 0.0 || df < delta)) delta = df;
        }
        bool ok = delta > 0.0 && getenv("TRIDSK_NO_LATTICE") == nullptr;
        int m = 0;
        const double nk2 = -(double)P.long_inv_two_sigma2 * 1.4426950408889634;
        for (int k = 0; k < n_types && ok; ++k) {
            if (k > 0) {
                const double df = (double)radius_h[ord[k]] - radius_h[ord[k - 1]];
                if (df <= 1e-6) { /* same m */ }
                else if (fabs(df - delta) <= 1e-5) { ++m; lat.step_mask |= 1u << k; }
                else ok = false;
            }
            // exact lattice point instead of the table value: the deviation allowed above is 1e-5 A
            if (fabs(((double)radius_h[ord[0]] + m * delta) - radius_h[ord[k]]) > 2e-5) ok = false;
            lat.order[k] = (unsigned char)ord[k];
            lat.cm[k] = (float)exp2(nk2 * (m * delta) * (m * delta));
        }
        if (ok && m * delta * 2.0 * fabs(nk2) * 12.0 < 60.0) {       // B^m stays far from overflow for |x| < 12 A
            lat.on = lat.step_mask == ((n_types >= 32 ? 0xffffffffu : ((1u << n_types) - 1u)) & ~1u) ? 2 : 1;
            lat.delta_k = (float)(-2.0 * nk2 * delta); lat.rmin = radius_h[ord[0]];
        }
    }
#define TRIDSK_GB_LAUNCH(NT)                                                                                              \
    do {                                                                                                                  \
        if (lat.on == 2) grid_build_kernel<NT, 2><<<g, GB_THREADS, 0, s>>>(rec, n_rec, tab, n_types, P, grid, dc_max, lat, rec_radius_dev, out);   \
        else if (lat.on) grid_build_kernel<NT, 1><<<g, GB_THREADS, 0, s>>>(rec, n_rec, tab, n_types, P, grid, dc_max, lat, rec_radius_dev, out);  \
        else grid_build_kernel<NT, 0><<<g, GB_THREADS, 0, s>>>(rec, n_rec, tab, n_types, P, grid, dc_max, lat, rec_radius_dev, out);            \
    } while (0)
    if (n_types <= 8) TRIDSK_GB_LAUNCH(8);
    else if (n_types <= 16) TRIDSK_GB_LAUNCH(16);
    else TRIDSK_GB_LAUNCH(32);
#undef TRIDSK_GB_LAUNCH
    return cudaGetLastError();
}

// ------------------------------------------------------------------ cell-packed copy of the grid (DGrid::gp)
// gp[t][z][y][x] = {g(x,y), g(x+1,y), g(x,y+1), g(x+1,y+1)} at the same (t, z); indices clamped at the upper
// edges (those records are never the base of a cell: i0 <= n - 2).  The 8 corners of a trilinear cell -- the xy
// quad of plane z and the quad of plane z + 1 -- are then ONE aligned 32-byte record (one L2 sector; one 256-bit load on
// sm_100), which is what the chain kernels gather.
__global__ void __launch_bounds__(256) grid_pack_kernel(const DGrid G, float4* __restrict__ out) {
    const size_t total = G.plane * (size_t)G.n_types;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % G.nx), y = (int)((i / G.nx) % G.ny);
        const int dx = (x + 1 < G.nx) ? 1 : 0;
        const size_t dy = (y + 1 < G.ny) ? (size_t)G.nx : 0;
        const int z = (int)((i / ((size_t)G.nx * G.ny)) % G.nz);
        const size_t dz = (z + 1 < G.nz) ? (size_t)G.nx * G.ny : 0;         // the record above (clamped at the top plane)
        out[2 * i] = make_float4(G.g[i], G.g[i + dx], G.g[i + dy], G.g[i + dy + dx]);
        out[2 * i + 1] = make_float4(G.g[i + dz], G.g[i + dz + dx], G.g[i + dz + dy], G.g[i + dz + dy + dx]);
    }
}

cudaError_t launch_grid_pack(cudaStream_t s, DGrid grid, float4* out) {
    const size_t total = grid.plane * (size_t)grid.n_types;
    const int blocks = (int)std::min<size_t>((total + 255) / 256, 148 * 16);
    grid_pack_kernel<<<blocks, 256, 0, s>>>(grid, out);
    return cudaGetLastError();
}
