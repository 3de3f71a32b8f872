// mdn.cu -- device-side preparation of the mixture-density term (tridsk_load_mdn; O15): bounding spheres of the residues
// and the packed parameter records.  Every value that the term's arithmetic uses is formed here, on the device, from the
// caller's plain (pi, mu, sigma): a = w_mdn pi / (sigma sqrt(2 pi)), nk2 = -log2(e) / (2 sigma^2), 1 / sigma^2 (mdn.cuh).
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

// One CTA per ligand: records [n_res][n][K] in the library's INTERNAL atom order from the caller's arrays in the
// caller's atom order (atom_i carries the original index of an internal atom).
__global__ void mdn_pack_kernel(const LigHdr* __restrict__ hdr, const int* __restrict__ atom_i, int n_res, int K,
                                const long long* __restrict__ lig_off, const float* __restrict__ pi, const float* __restrict__ mu,
                                const float* __restrict__ sigma, float w_mdn, float4* __restrict__ par, int* __restrict__ bad) {
    const int lig = blockIdx.x;
    const LigHdr h = hdr[lig];
    const long long base = lig_off[lig];
    const long long total = (long long)n_res * h.n * K;
    for (long long e = threadIdx.x; e < total; e += blockDim.x) {
        const int k = (int)(e % K);
        const long long ip = e / K;
        const int p = (int)(ip % h.n);
        const long long i = ip / h.n;
        const int orig = (atom_i[h.atom_off + p] >> 16) & 0xff;
        const long long src = base + (i * h.n + orig) * K + k;
        const float sg = sigma[src], w = pi[src], m = mu[src];
        if (!(sg > 0.f) || !isfinite(sg) || !isfinite(w) || !isfinite(m)) { *bad = 1; par[base + e] = make_float4(0.f, 0.f, 0.f, 0.f); continue; }
        const float inv_s2 = 1.f / (sg * sg);
        par[base + e] = make_float4(w_mdn * w / (sg * 2.5066282746310002f), m, -0.7213475204444817f * inv_s2, inv_s2);
    }
}

cudaError_t launch_mdn_spheres(cudaStream_t s, const float* res_xyz, const int* res_off, int n_res, float d_cut, float4* rec, float4* sph) {
    if (n_res <= 0) return cudaSuccess;
    mdn_sphere_kernel<<<(n_res + 127) / 128, 128, 0, s>>>(res_xyz, res_off, n_res, d_cut, rec, sph);
    return cudaGetLastError();
}

cudaError_t launch_mdn_pack(cudaStream_t s, const LigHdr* hdr, const int* atom_i, int n_lig, int n_res, int K, const long long* lig_off,
                            const float* pi, const float* mu, const float* sigma, float w_mdn, float4* par, int* bad) {
    if (n_lig <= 0 || n_res <= 0) return cudaSuccess;
    mdn_pack_kernel<<<n_lig, 256, 0, s>>>(hdr, atom_i, n_res, K, lig_off, pi, mu, sigma, w_mdn, par, bad);
    return cudaGetLastError();
}
