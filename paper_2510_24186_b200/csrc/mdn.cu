// mdn.cu -- device-side preparation of the mixture-density term (tridsk_load_mdn; O15): bounding spheres of the residues
// and the packed parameter records.  Every value that the term's arithmetic uses is formed here, on the device, from the
// caller's plain (pi, mu, sigma): a = w_mdn pi / (sigma sqrt(2 pi)), nk2 = -log2(e) / (2 sigma^2) (mdn.cuh).
#include "internal.h"

// One thread per residue: copy its atoms into float4 records and take the bounding sphere about their centroid.
__global__ void mdn_sphere_kernel(const float* __restrict__ res_xyz, const int* __restrict__ res_off, int n_res, float d_cut,
                                  float4* __restrict__ rec, float4* __restrict__ sph) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_res) return;
    const int r0 = res_off[i], r1 = res_off[i + 1];
    float cx = 0.f, cy = 0.f, cz = 0.f;
    for (int r = r0; r < r1; ++r) {
        const float x = res_xyz[3 * r], y = res_xyz[3 * r + 1], z = res_xyz[3 * r + 2];
        rec[r] = make_float4(x, y, z, 0.f);
        cx += x; cy += y; cz += z;
    }
    const float inv = r1 > r0 ? 1.f / (float)(r1 - r0) : 0.f;
    cx *= inv; cy *= inv; cz *= inv;
    float rad2 = 0.f;
    for (int r = r0; r < r1; ++r) {
        const float dx = res_xyz[3 * r] - cx, dy = res_xyz[3 * r + 1] - cy, dz = res_xyz[3 * r + 2] - cz;
        rad2 = fmaxf(rad2, dx * dx + dy * dy + dz * dz);
    }
    const float reach = (r1 > r0) ? sqrtf(rad2) * 1.0001f + d_cut + 1e-4f : -1.f;   // an empty residue is never visited
    sph[i] = make_float4(cx, cy, cz, reach > 0.f ? reach * reach : -1.f);
}

// One CTA per ligand: parameter slots [n_res][n][K4 float4] (internal.h: blocks of ten components {a, mu, nk2}, unused floats
// zero) in the library's INTERNAL atom order from the caller's arrays [n_res][n][K] in the caller's atom order (atom_i carries
// the original index of an internal atom).  lig_off / in_off: start of the ligand's block in par / in the caller's arrays.
__global__ void mdn_pack_kernel(const LigHdr* __restrict__ hdr, const int* __restrict__ atom_i, int n_res, int K,
                                const long long* __restrict__ lig_off, const long long* __restrict__ in_off,
                                const float* __restrict__ pi, const float* __restrict__ mu,
                                const float* __restrict__ sigma, float w_mdn, float4* __restrict__ par, int* __restrict__ bad) {
    const int lig = blockIdx.x;
    const LigHdr h = hdr[lig];
    const int K4 = mdn_slot_f4(K);
    const long long base = lig_off[lig], ibase = in_off[lig];
    const long long total = (long long)n_res * h.n * K4;
    for (long long e = threadIdx.x; e < total; e += blockDim.x) {
        const int f4 = (int)(e % K4);
        const long long ip = e / K4;
        const int p = (int)(ip % h.n);
        const long long i = ip / h.n;
        const int orig = (atom_i[h.atom_off + p] >> 16) & 0xff;
        float v[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int f = 4 * f4 + c, w = f & 31, k = 10 * (f >> 5) + w / 3, fld = w % 3;
            v[c] = 0.f;
            if (w >= 30 || k >= K) continue;
            const long long src = ibase + (i * h.n + orig) * K + k;
            const float sg = sigma[src], wt = pi[src], m = mu[src];
            if (!(sg > 0.f) || !isfinite(sg) || !isfinite(wt) || !isfinite(m)) { *bad = 1; continue; }
            v[c] = fld == 0 ? w_mdn * wt / (sg * 2.5066282746310002f) : fld == 1 ? m : -0.7213475204444817f / (sg * sg);
        }
        par[base + e] = make_float4(v[0], v[1], v[2], v[3]);
    }
}

cudaError_t launch_mdn_spheres(cudaStream_t s, const float* res_xyz, const int* res_off, int n_res, float d_cut, float4* rec, float4* sph) {
    if (n_res <= 0) return cudaSuccess;
    mdn_sphere_kernel<<<(n_res + 127) / 128, 128, 0, s>>>(res_xyz, res_off, n_res, d_cut, rec, sph);
    return cudaGetLastError();
}

cudaError_t launch_mdn_pack(cudaStream_t s, const LigHdr* hdr, const int* atom_i, int n_lig, int n_res, int K, const long long* lig_off,
                            const long long* in_off, const float* pi, const float* mu, const float* sigma, float w_mdn, float4* par, int* bad) {
    if (n_lig <= 0 || n_res <= 0) return cudaSuccess;
    mdn_pack_kernel<<<n_lig, 256, 0, s>>>(hdr, atom_i, n_res, K, lig_off, in_off, pi, mu, sigma, w_mdn, par, bad);
    return cudaGetLastError();
}

// One thread per cell of the cell list: the receptor atoms within d_cut + half a cell diagonal of the cell's centre, in
// (residue, atom index) order; the first entry of a residue's run carries residue id | run length << 16 in w, the second
// the same header of the NEXT run of the cell (-1: none), the others the residue id; runs are padded to an even length (32-byte alignment for 256-bit loads).  fill = false: counts[c] = how many; fill = true: written to cell_at[off[c] ..].
__global__ void mdn_cell_kernel(MdnDev M, float cell, bool fill, int* __restrict__ counts_or_off, float4* __restrict__ cell_at) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    const int ncell = M.nc[0] * M.nc[1] * M.nc[2];
    if (c >= ncell) return;
    const int ix = c % M.nc[0], iy = (c / M.nc[0]) % M.nc[1], iz = c / (M.nc[0] * M.nc[1]);
    const float x = M.glo[0] + cell * ((float)ix + 0.5f), y = M.glo[1] + cell * ((float)iy + 0.5f), z = M.glo[2] + cell * ((float)iz + 0.5f);
    const float half_diag = 0.8660254f * cell;
    const float reach = M.d_cut + half_diag * 1.001f + 1e-3f, reach2 = reach * reach;
    int n = 0, prev = -1;
    float4* dst = fill ? cell_at + counts_or_off[c] : nullptr;
    for (int i = 0; i < M.n_res; ++i) {
        const float4 s = M.sph[i];
        if (s.w < 0.f) continue;
        const float sx = x - s.x, sy = y - s.y, sz = z - s.z;
        const float lim = sqrtf(s.w) + half_diag;                 // grown bounding sphere + the cell's own radius
        if (sx * sx + sy * sy + sz * sz >= lim * lim) continue;
        const int first = n;
        for (int r = M.res_off[i]; r < M.res_off[i + 1]; ++r) {
            const float4 a = M.rec[r];
            const float dx = x - a.x, dy = y - a.y, dz = z - a.z;
            if (dx * dx + dy * dy + dz * dz < reach2) {
                if (fill) dst[n] = make_float4(a.x, a.y, a.z, __int_as_float(i));
                ++n;
            }
        }
        if ((n - first) & 1) {                                    // pad the run to an even length: an entry that can never be the minimum
            if (fill) dst[n] = make_float4(1e18f, 1e18f, 1e18f, __int_as_float(i));
            ++n;
        }
        if (fill && n > first) {
            const int hdr = i | ((n - first) << 16);
            dst[first].w = __int_as_float(hdr);
            dst[first + 1].w = __int_as_float(-1);                  // the next run's header goes here (-1: this is the last run)
            if (prev >= 0) dst[prev + 1].w = __int_as_float(hdr);
            prev = first;
        }
    }
    if (!fill) counts_or_off[c] = n;
}

cudaError_t launch_mdn_cells(cudaStream_t s, const MdnDev& M, float cell, bool fill, int* counts_or_off, float4* cell_at) {
    const int ncell = M.nc[0] * M.nc[1] * M.nc[2];
    if (ncell <= 0) return cudaSuccess;
    mdn_cell_kernel<<<(ncell + 127) / 128, 128, 0, s>>>(M, cell, fill, counts_or_off, cell_at);
    return cudaGetLastError();
}

// One thread per cell: walk the cell's stream run by run.  fill = false: counts[c] = number of runs; fill = true: the
// directory entries {header, position in cell_at} written to dir[off[c] ..].
__global__ void mdn_dir_kernel(MdnDev M, bool fill, int* __restrict__ counts_or_off, int2* __restrict__ dir) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    const int ncell = M.nc[0] * M.nc[1] * M.nc[2];
    if (c >= ncell) return;
    const int e1 = M.cell_off[c + 1];
    int n = 0;
    int2* dst = fill ? dir + counts_or_off[c] : nullptr;
    for (int en = M.cell_off[c]; en < e1;) {
        const int hdr = __float_as_int(M.cell_at[en].w);
        if (fill) dst[n] = make_int2(hdr, en);
        ++n;
        en += hdr >> 16;
    }
    if (!fill) counts_or_off[c] = n;
}

cudaError_t launch_mdn_dir(cudaStream_t s, const MdnDev& M, bool fill, int* counts_or_off, int2* dir) {
    const int ncell = M.nc[0] * M.nc[1] * M.nc[2];
    if (ncell <= 0) return cudaSuccess;
    mdn_dir_kernel<<<(ncell + 127) / 128, 128, 0, s>>>(M, fill, counts_or_off, dir);
    return cudaGetLastError();
}
