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

cudaError_t launch_topk(cudaStream_t s, const TopkLaunch& a) {
    if (a.n_lig <= 0 || a.top_k <= 0) return cudaSuccess;
    topk_kernel<<<a.n_lig, TOPK_THREADS, 0, s>>>(a);
    return cudaGetLastError();
}
