// topk.cu -- hot-path step a9 (O13): per ligand, the top_k lowest per-chain best energies across chains,
// ties broken by the lower chain id ("ranked ... top N conformations"), plus the E_screen epilogue
// E_dock / (1 + w_tor * N_tor).  One CTA per ligand; k rounds of a lexicographic (E, chain) arg-min
// strictly above the previous pick -- deterministic, any n_chains, O(k * n_chains / 256) per thread.
#include "internal.h"

#define TOPK_THREADS 256

__device__ __forceinline__ bool lex_less(float ea, int ia, float eb, int ib) { return ea < eb || (ea == eb && ia < ib); }

__global__ void __launch_bounds__(TOPK_THREADS) topk_kernel(const TopkLaunch a) {
    __shared__ float s_e[TOPK_THREADS / 32];
    __shared__ int s_i[TOPK_THREADS / 32];
    __shared__ float s_pe;
    __shared__ int s_pi;
    const int lig = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float* e = a.e_best + (size_t)lig * a.n_chains;
    const int T = a.hdr[lig].T;
    float pe = -INFINITY;      // previous pick (exclusive lower bound)
    int pi = -1;
    for (int r = 0; r < a.top_k; ++r) {
        float be = INFINITY;
        int bi = 0x7fffffff;
        for (int c = tid; c < a.n_chains; c += TOPK_THREADS) {
            float v = e[c];
            if (!(v == v)) v = INFINITY;                       // NaN energies sort last
            if (lex_less(pe, pi, v, c) && lex_less(v, c, be, bi)) { be = v; bi = c; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float oe = __shfl_xor_sync(0xffffffffu, be, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (lex_less(oe, oi, be, bi)) { be = oe; bi = oi; }
        }
        if (lane == 0) { s_e[warp] = be; s_i[warp] = bi; }
        __syncthreads();
        if (tid == 0) {
            for (int w = 1; w < TOPK_THREADS / 32; ++w)
                if (lex_less(s_e[w], s_i[w], be, bi)) { be = s_e[w]; bi = s_i[w]; }
            s_pe = be; s_pi = bi;
            const size_t o = (size_t)lig * a.top_k + r;
            const float ed = e[bi];
            a.out_energy[2 * o] = ed;
            a.out_energy[2 * o + 1] = ed / (1.f + a.w_tor * (float)T);
            a.out_chain[o] = bi;
        }
        __syncthreads();
        pe = s_pe; pi = s_pi;
        const float* src = a.pose_best + ((size_t)lig * a.n_chains + pi) * a.pose_stride;
        float* dst = a.out_pose + ((size_t)lig * a.top_k + r) * a.pose_stride;
        for (int i = tid; i < a.pose_stride; i += TOPK_THREADS) dst[i] = src[i];
    }
}


// ------------------------------------------------------------------ O14: duplicate-removing top-k (reading G20)
// "Ranked ... clustered to remove the duplicates ... top N": walk the chains in the order of O13; a chain's best pose is a
// duplicate if its heavy-atom RMSD (same atom order, no superposition -- poses live in the receptor frame) to an already
// kept pose is below cluster_rmsd, otherwise it is kept; stop at top_k kept.  Slots that cannot be filled get chain -1,
// energies +inf and a zero pose.  One CTA per ligand; the candidate's coordinates come from a forward-kinematics pass in
// this kernel (O8: fragment frames composed from the root down, one thread per fragment).
__global__ void __launch_bounds__(TOPK_THREADS) topk_cluster_kernel(const TopkLaunch a) {
    extern __shared__ __align__(16) float cl_smem[];
    __shared__ float s_e[TOPK_THREADS / 32];
    __shared__ int s_i[TOPK_THREADS / 32];
    __shared__ float s_pe;
    __shared__ int s_pi, s_dup;
    const int lig = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const LigHdr h = a.hdr[lig];
    const int n = h.n, T = h.T;
    float* kept = cl_smem;                                   // [top_k][3 n]
    float* cand = kept + (size_t)a.top_k * 3 * a.max_atoms;  // [3 n]
    const float* e = a.e_best + (size_t)lig * a.n_chains;
    const float4* ref = a.atom_f4 + h.atom_off;
    const LaneFrag* frag = a.lane_frags + h.frag_off;
    const float thr2 = a.cluster_rmsd * a.cluster_rmsd * (float)n;   // compare the SUM of squared deviations
    float pe = -INFINITY;
    int pi = -1, n_kept = 0;
    for (int it = 0; it < a.n_chains && n_kept < a.top_k; ++it) {
        // next chain in (E, chain) order
        float be = INFINITY;
        int bi = 0x7fffffff;
        for (int c = tid; c < a.n_chains; c += TOPK_THREADS) {
            float v = e[c];
            if (!(v == v)) v = INFINITY;
            if (lex_less(pe, pi, v, c) && lex_less(v, c, be, bi)) { be = v; bi = c; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float oe = __shfl_xor_sync(0xffffffffu, be, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (lex_less(oe, oi, be, bi)) { be = oe; bi = oi; }
        }
        if (lane == 0) { s_e[warp] = be; s_i[warp] = bi; }
        __syncthreads();
        if (tid == 0) {
            for (int w = 1; w < TOPK_THREADS / 32; ++w)
                if (lex_less(s_e[w], s_i[w], be, bi)) { be = s_e[w]; bi = s_i[w]; }
            s_pe = be; s_pi = bi; s_dup = 0;
        }
        __syncthreads();
        pe = s_pe; pi = s_pi;
        const float* pose = a.pose_best + ((size_t)lig * a.n_chains + pi) * a.pose_stride;
        // a3 / O8: thread g composes the frame of fragment g along its ancestors and places the fragment's own atoms
        if (tid <= T) {
            int path[TRIDSK_MAX_TORSIONS + 1], np_ = 0;
            for (int g = tid; g > 0; g = frag[g].parent) path[np_++] = g;
            float q[4] = {pose[3], pose[4], pose[5], pose[6]};
            const float qn = rsqrtf(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
            const float w = q[0] * qn, x = q[1] * qn, y = q[2] * qn, z = q[3] * qn;
            float R[9] = {1.f - 2.f * (y * y + z * z), 2.f * (x * y - w * z), 2.f * (x * z + w * y),
                          2.f * (x * y + w * z), 1.f - 2.f * (x * x + z * z), 2.f * (y * z - w * x),
                          2.f * (x * z - w * y), 2.f * (y * z + w * x), 1.f - 2.f * (x * x + y * y)};
            float p[3] = {pose[0], pose[1], pose[2]};
            for (int k = np_ - 1; k >= 0; --k) {
                const LaneFrag f = frag[path[k]];
                float sn, cs;
                sincosf(pose[7 + f.tor], &sn, &cs);
                const float oc = 1.f - cs;
                float Lm[9];
                Lm[0] = fmaf(oc * f.ux, f.ux, cs);         Lm[1] = fmaf(oc * f.ux, f.uy, -sn * f.uz); Lm[2] = fmaf(oc * f.ux, f.uz, sn * f.uy);
                Lm[3] = fmaf(oc * f.uy, f.ux, sn * f.uz);  Lm[4] = fmaf(oc * f.uy, f.uy, cs);         Lm[5] = fmaf(oc * f.uy, f.uz, -sn * f.ux);
                Lm[6] = fmaf(oc * f.uz, f.ux, -sn * f.uy); Lm[7] = fmaf(oc * f.uz, f.uy, sn * f.ux);  Lm[8] = fmaf(oc * f.uz, f.uz, cs);
                const float c0 = f.ox - (Lm[0] * f.ox + Lm[1] * f.oy + Lm[2] * f.oz);
                const float c1 = f.oy - (Lm[3] * f.ox + Lm[4] * f.oy + Lm[5] * f.oz);
                const float c2 = f.oz - (Lm[6] * f.ox + Lm[7] * f.oy + Lm[8] * f.oz);
                float Rn[9], pn[3];
#pragma unroll
                for (int r = 0; r < 3; ++r) {
                    Rn[3 * r + 0] = R[3 * r] * Lm[0] + R[3 * r + 1] * Lm[3] + R[3 * r + 2] * Lm[6];
                    Rn[3 * r + 1] = R[3 * r] * Lm[1] + R[3 * r + 1] * Lm[4] + R[3 * r + 2] * Lm[7];
                    Rn[3 * r + 2] = R[3 * r] * Lm[2] + R[3 * r + 1] * Lm[5] + R[3 * r + 2] * Lm[8];
                    pn[r] = R[3 * r] * c0 + R[3 * r + 1] * c1 + R[3 * r + 2] * c2 + p[r];
                }
#pragma unroll
                for (int i = 0; i < 9; ++i) R[i] = Rn[i];
#pragma unroll
                for (int i = 0; i < 3; ++i) p[i] = pn[i];
            }
            const LaneFrag me = frag[tid];
            for (int at = me.lo; at < me.own_hi; ++at) {
                const float4 r = ref[at];
                cand[3 * at] = R[0] * r.x + R[1] * r.y + R[2] * r.z + p[0];
                cand[3 * at + 1] = R[3] * r.x + R[4] * r.y + R[5] * r.z + p[1];
                cand[3 * at + 2] = R[6] * r.x + R[7] * r.y + R[8] * r.z + p[2];
            }
        }
        __syncthreads();
        // squared deviation to every kept pose: warp w takes kept poses w, w + 8, ...
        for (int j = warp; j < n_kept; j += TOPK_THREADS / 32) {
            const float* kx = kept + (size_t)j * 3 * a.max_atoms;
            float sd = 0.f;
            for (int i = lane; i < 3 * n; i += 32) { const float d = cand[i] - kx[i]; sd = fmaf(d, d, sd); }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) sd += __shfl_xor_sync(0xffffffffu, sd, o);
            if (lane == 0 && sd < thr2) s_dup = 1;
        }
        __syncthreads();
        if (!s_dup) {                                        // uniform
            float* kx = kept + (size_t)n_kept * 3 * a.max_atoms;
            for (int i = tid; i < 3 * n; i += TOPK_THREADS) kx[i] = cand[i];
            const size_t o = (size_t)lig * a.top_k + n_kept;
            if (tid == 0) {
                const float ed = e[pi];
                a.out_energy[2 * o] = ed;
                a.out_energy[2 * o + 1] = ed / (1.f + a.w_tor * (float)T);
                a.out_chain[o] = pi;
            }
            float* dst = a.out_pose + o * a.pose_stride;
            for (int i = tid; i < a.pose_stride; i += TOPK_THREADS) dst[i] = pose[i];
            ++n_kept;
        }
        __syncthreads();
    }
    for (int r = n_kept; r < a.top_k; ++r) {                 // fewer clusters than top_k
        const size_t o = (size_t)lig * a.top_k + r;
        if (tid == 0) { a.out_energy[2 * o] = INFINITY; a.out_energy[2 * o + 1] = INFINITY; a.out_chain[o] = -1; }
        float* dst = a.out_pose + o * a.pose_stride;
        for (int i = tid; i < a.pose_stride; i += TOPK_THREADS) dst[i] = 0.f;
    }
}

size_t topk_cluster_smem(int top_k, int max_atoms, int max_tor) {
    (void)max_tor;
    return sizeof(float) * 3 * (size_t)max_atoms * ((size_t)top_k + 1);
}

// per device (function attributes are per device): called by tridsk_create
cudaError_t topk_prepare() {
    return cudaFuncSetAttribute(topk_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TRIDSK_SMEM_MAX_CTA - 2048);
}

cudaError_t launch_topk(cudaStream_t s, const TopkLaunch& a) {
    if (a.n_lig <= 0 || a.top_k <= 0) return cudaSuccess;
    if (a.cluster_rmsd > 0.f) {
        const size_t smem = topk_cluster_smem(a.top_k, a.max_atoms, a.max_tor);
        if (smem > TRIDSK_SMEM_MAX_CTA - 2048) return cudaErrorInvalidValue;
        topk_cluster_kernel<<<a.n_lig, TOPK_THREADS, smem, s>>>(a);
    } else {
        topk_kernel<<<a.n_lig, TOPK_THREADS, 0, s>>>(a);
    }
    return cudaGetLastError();
}
