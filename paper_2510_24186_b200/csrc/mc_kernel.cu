// mc_kernel.cu -- the fused per-chain Monte Carlo kernel (steps a1..a8, a10) and the pose-evaluation
// kernel behind tridsk_score_grad (a3..a6).  One warp per chain / pose; see chain.cuh.
#include "chain.cuh"

// ------------------------------------------------------------------ chain state I/O (once per launch)
__device__ __forceinline__ void load_pose(const float* __restrict__ src, int T, float t[3], float q[4], float& th) {
    const int lane = threadIdx.x & 31;
    t[0] = src[0]; t[1] = src[1]; t[2] = src[2];
    q[0] = src[3]; q[1] = src[4]; q[2] = src[5]; q[3] = src[6];
    th = (lane >= 1 && lane <= T) ? src[6 + lane] : 0.f;
}
__device__ __forceinline__ void store_pose(float* __restrict__ dst, int T, int stride, const float t[3], const float q[4], float th) {
    const int lane = threadIdx.x & 31;
    if (lane == 0) {
        dst[0] = t[0]; dst[1] = t[1]; dst[2] = t[2];
        dst[3] = q[0]; dst[4] = q[1]; dst[5] = q[2]; dst[6] = q[3];
    } else if (lane <= T) dst[6 + lane] = th;
    for (int e = 7 + T + lane; e < stride; e += 32) dst[e] = 0.f;
}

// ------------------------------------------------------------------ the fused MC kernel
template <int J, bool MDN>
__global__ void __launch_bounds__(TRIDSK_WARPS_PER_CTA * 32) mc_kernel(const McLaunch a) {
    __shared__ float sP_all[TRIDSK_WARPS_PER_CTA][6 * J * 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int bpl = (a.n_chains + TRIDSK_WARPS_PER_CTA - 1) / TRIDSK_WARPS_PER_CTA;
    const int chain = (blockIdx.x % bpl) * TRIDSK_WARPS_PER_CTA + warp;
    if (chain >= a.n_chains) return;
    const int lig = a.lig_list[blockIdx.x / bpl];
    float* sP = sP_all[warp];

    Lig<J> L;
    load_lig<J>(L, a.hdr, a.atom_f4, a.atom_i, a.frags, a.rounds, lig);
    const DParams& P = a.P;
    const int T = L.T;
    const float4* mdn_par = a.mdn.n_res > 0 ? a.mdn.par + a.mdn.lig_off[lig] : nullptr;
    const size_t cidx = (size_t)lig * a.n_chains + chain;
    const uint2 key = make_uint2((uint32_t)a.seed, (uint32_t)(a.seed >> 32));
    const uint32_t gchain = (uint32_t)(a.chain_base + chain);      // Philox counter word 0

    float ct[3], cq[4], cth, ecur;          // current accepted state
    float bt[3], bq[4], bth, ebest;         // best state seen
    float x[J], y[J], z[J];
    float gt[3], gw[3], gth;

    if (a.init_mode == 2) {                 // resume
        load_pose(a.pose_cur + cidx * a.pose_stride, T, ct, cq, cth);
        load_pose(a.pose_best + cidx * a.pose_stride, T, bt, bq, bth);
        ecur = a.e_cur[cidx]; ebest = a.e_best[cidx];
    } else {
        if (a.init_mode == 1) {
            load_pose(a.init_poses + cidx * a.pose_stride, T, ct, cq, cth);
            quat_normalise(cq);
        } else {                            // a1 / O11: Philox initialisation; lane l computes block purpose 2 + l
            const uint4 r = philox4x32_10(make_uint4(gchain, 0u, (uint32_t)(a.lig_base + lig), 2u + (uint32_t)lane), key);
            const float u0 = u01(r.x), u1 = u01(r.y), u2 = u01(r.z), u3 = u01(r.w);
            const float a0 = __shfl_sync(FULL_MASK, u0, 0), a1 = __shfl_sync(FULL_MASK, u1, 0), a2 = __shfl_sync(FULL_MASK, u2, 0);
            const float b0 = __shfl_sync(FULL_MASK, u0, 1), b1 = __shfl_sync(FULL_MASK, u1, 1), b2 = __shfl_sync(FULL_MASK, u2, 1);
            const float rr = a.radius * cbrtf(a0), zz = 2.f * a1 - 1.f, sq = sqrtf(fmaxf(1.f - zz * zz, 0.f));
            float sn, cs;
            sincosf(2.f * PI_F * a2, &sn, &cs);
            ct[0] = a.centre[0] + rr * sq * cs; ct[1] = a.centre[1] + rr * sq * sn; ct[2] = a.centre[2] + rr * zz;
            const float s1 = sqrtf(1.f - b0), s2 = sqrtf(b0);
            float sn1, cs1, sn2, cs2;
            sincosf(2.f * PI_F * b1, &sn1, &cs1);
            sincosf(2.f * PI_F * b2, &sn2, &cs2);
            cq[0] = s2 * cs2; cq[1] = s1 * sn1; cq[2] = s1 * cs1; cq[3] = s2 * sn2;
            quat_normalise(cq);
            // torsion k = f-1 takes element k%4 of block 4 + k/4, i.e. of lane 2 + k/4
            const int k = lane - 1, src = 2 + (k >> 2);
            const float v0 = __shfl_sync(FULL_MASK, u0, src & 31), v1 = __shfl_sync(FULL_MASK, u1, src & 31);
            const float v2 = __shfl_sync(FULL_MASK, u2, src & 31), v3 = __shfl_sync(FULL_MASK, u3, src & 31);
            const float uu = (k & 3) == 0 ? v0 : (k & 3) == 1 ? v1 : (k & 3) == 2 ? v2 : v3;
            cth = (lane >= 1 && lane <= T) ? PI_F * (2.f * uu - 1.f) : 0.f;
        }
        float ei, ea;
        eval_pose<J, false, MDN>(L, a.grid, P, a.mdn, mdn_par, a.rec, ct, cq, cth, x, y, z, ei, ea, gt, gw, gth, sP);
        ecur = warp_sum(ei + ea);
        ebest = ecur;
#pragma unroll
        for (int i = 0; i < 3; ++i) bt[i] = ct[i];
#pragma unroll
        for (int i = 0; i < 4; ++i) bq[i] = cq[i];
        bth = cth;
    }

    for (int s = 0; s < a.n_steps; ++s) {
        const uint32_t step = (uint32_t)(a.first_step + s);
        // O10: even lanes draw the perturbation block (purpose 0), odd lanes the Metropolis block (purpose 1)
        const uint4 r = philox4x32_10(make_uint4(gchain, step, (uint32_t)(a.lig_base + lig), (uint32_t)(lane & 1)), key);
        const float u0 = __shfl_sync(FULL_MASK, u01(r.x), 0), u1 = __shfl_sync(FULL_MASK, u01(r.y), 0);
        const float u2 = __shfl_sync(FULL_MASK, u01(r.z), 0), u3 = __shfl_sync(FULL_MASK, u01(r.w), 0);
        const float um = __shfl_sync(FULL_MASK, u01(r.x), 1);

        // a2 / O12: perturb one entity of {translation, rotation, torsion k}
        float pt[3] = {ct[0], ct[1], ct[2]}, pq[4] = {cq[0], cq[1], cq[2], cq[3]}, pth = cth;
        const int entity = min((int)(u0 * (float)(T + 2)), T + 1);
        if (entity == 0) {
            pt[0] = fminf(fmaxf(pt[0] + P.pert_trans * (2.f * u1 - 1.f), a.box_min[0]), a.box_max[0]);
            pt[1] = fminf(fmaxf(pt[1] + P.pert_trans * (2.f * u2 - 1.f), a.box_min[1]), a.box_max[1]);
            pt[2] = fminf(fmaxf(pt[2] + P.pert_trans * (2.f * u3 - 1.f), a.box_min[2]), a.box_max[2]);
        } else if (entity == 1) {
            quat_rotate_by(pq, P.pert_rot * (2.f * u1 - 1.f), P.pert_rot * (2.f * u2 - 1.f), P.pert_rot * (2.f * u3 - 1.f));
        } else if (lane == entity - 1) {
            pth = PI_F * (2.f * u1 - 1.f);
        }

        // a3..a7: n_refine Adam steps on the 6+T tangent components (moments reset every MC step, G12)
        float m[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, v[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        float b1p = 1.f, b2p = 1.f;
        for (int rf = 0; rf < P.n_refine; ++rf) {
            float ei, ea;
            eval_pose<J, true, MDN>(L, a.grid, P, a.mdn, mdn_par, a.rec, pt, pq, pth, x, y, z, ei, ea, gt, gw, gth, sP);
            b1p *= P.adam_b1; b2p *= P.adam_b2;
            const float c1 = __fdividef(1.f, 1.f - b1p), c2 = __fdividef(1.f, 1.f - b2p);   // 2-ulp division / square root:
            // far inside the tolerance, and the IEEE forms are slow-path subroutines on the chain's critical path
            float g[7] = {gt[0], gt[1], gt[2], gw[0], gw[1], gw[2], gth}, dl[7];
#pragma unroll
            for (int i = 0; i < 7; ++i) {
                m[i] = P.adam_b1 * m[i] + (1.f - P.adam_b1) * g[i];
                v[i] = P.adam_b2 * v[i] + (1.f - P.adam_b2) * g[i] * g[i];
                dl[i] = __fdividef(-P.lr * (m[i] * c1), sqrt_approx(v[i] * c2) + P.adam_eps);
            }
            pt[0] = fminf(fmaxf(pt[0] + dl[0], a.box_min[0]), a.box_max[0]);
            pt[1] = fminf(fmaxf(pt[1] + dl[1], a.box_min[1]), a.box_max[1]);
            pt[2] = fminf(fmaxf(pt[2] + dl[2], a.box_min[2]), a.box_max[2]);
            quat_rotate_by(pq, dl[3], dl[4], dl[5]);
            float th = pth + dl[6];
            if (th >= PI_F) th -= 2.f * PI_F;
            if (th < -PI_F) th += 2.f * PI_F;
            pth = (lane >= 1 && lane <= T) ? th : 0.f;
        }

        // a8: energy of the refined proposal, Metropolis, best tracking
        float ei, ea;
        eval_pose<J, false, MDN>(L, a.grid, P, a.mdn, mdn_par, a.rec, pt, pq, pth, x, y, z, ei, ea, gt, gw, gth, sP);
        const float enew = warp_sum(ei + ea);
        const bool accept = isfinite(enew) && (um < expf(-P.beta * (enew - ecur)));
        if (a.trace != nullptr && lane == 0) {
            tridsk_trace_rec rec;
            rec.e_prop = enew; rec.e_cur = ecur; rec.u = um; rec.flags = (accept ? 1 : 0) | (entity << 8);
            a.trace[cidx * a.trace_stride + a.trace_off + s] = rec;
        }
        if (accept) {
#pragma unroll
            for (int i = 0; i < 3; ++i) ct[i] = pt[i];
#pragma unroll
            for (int i = 0; i < 4; ++i) cq[i] = pq[i];
            cth = pth; ecur = enew;
            if (enew < ebest) {
#pragma unroll
                for (int i = 0; i < 3; ++i) bt[i] = pt[i];
#pragma unroll
                for (int i = 0; i < 4; ++i) bq[i] = pq[i];
                bth = pth; ebest = enew;
            }
        }
    }

    store_pose(a.pose_cur + cidx * a.pose_stride, T, a.pose_stride, ct, cq, cth);
    store_pose(a.pose_best + cidx * a.pose_stride, T, a.pose_stride, bt, bq, bth);
    if (lane == 0) { a.e_cur[cidx] = ecur; a.e_best[cidx] = ebest; }
}

cudaError_t launch_mc(cudaStream_t s, int J, const McLaunch& a) {
    const int bpl = (a.n_chains + TRIDSK_WARPS_PER_CTA - 1) / TRIDSK_WARPS_PER_CTA;
    const long long blocks = (long long)a.n_list * bpl;
    if (blocks <= 0) return cudaSuccess;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    const dim3 grid((unsigned)blocks), block(TRIDSK_WARPS_PER_CTA * 32);
    if (a.mdn.n_res > 0) {
        switch (J) {
            case 1: mc_kernel<1, true><<<grid, block, 0, s>>>(a); break;
            case 2: mc_kernel<2, true><<<grid, block, 0, s>>>(a); break;
            case 3: mc_kernel<3, true><<<grid, block, 0, s>>>(a); break;
            case 4: mc_kernel<4, true><<<grid, block, 0, s>>>(a); break;
            default: return cudaErrorInvalidValue;
        }
    } else {
        switch (J) {
            case 1: mc_kernel<1, false><<<grid, block, 0, s>>>(a); break;
            case 2: mc_kernel<2, false><<<grid, block, 0, s>>>(a); break;
            case 3: mc_kernel<3, false><<<grid, block, 0, s>>>(a); break;
            case 4: mc_kernel<4, false><<<grid, block, 0, s>>>(a); break;
            default: return cudaErrorInvalidValue;
        }
    }
    return cudaGetLastError();
}

// ------------------------------------------------------------------ tridsk_score_grad: one warp per pose
template <int J, bool MDN>
__device__ __forceinline__ void score_one(const ScoreLaunch& a, int i, int lig, float* sP) {
    const int lane = threadIdx.x & 31;
    Lig<J> L;
    load_lig<J>(L, a.hdr, a.atom_f4, a.atom_i, a.frags, a.rounds, lig);
    float t[3], q[4], th, x[J], y[J], z[J], gt[3], gw[3], gth, ei, ea;
    load_pose(a.poses + (size_t)i * a.pose_stride, L.T, t, q, th);
    quat_normalise(q);
    const float4* mdn_par = a.mdn.n_res > 0 ? a.mdn.par + a.mdn.lig_off[lig] : nullptr;
    RecDev no_rec;
    no_rec.atoms = nullptr;
    if (a.grad != nullptr) eval_pose<J, true, MDN>(L, a.grid, a.P, a.mdn, mdn_par, no_rec, t, q, th, x, y, z, ei, ea, gt, gw, gth, sP);
    else eval_pose<J, false, MDN>(L, a.grid, a.P, a.mdn, mdn_par, no_rec, t, q, th, x, y, z, ei, ea, gt, gw, gth, sP);
    ei = warp_sum(ei); ea = warp_sum(ea);
    if (lane == 0) {
        a.energy[3 * (size_t)i] = ei + ea; a.energy[3 * (size_t)i + 1] = ei; a.energy[3 * (size_t)i + 2] = ea;
    }
    if (a.grad != nullptr) {
        float* g = a.grad + (size_t)i * a.grad_stride;
        if (lane == 0) { g[0] = gt[0]; g[1] = gt[1]; g[2] = gt[2]; g[3] = gw[0]; g[4] = gw[1]; g[5] = gw[2]; }
        else if (lane <= L.T) g[5 + lane] = gth;
        for (int e = 6 + L.T + lane; e < a.grad_stride; e += 32) g[e] = 0.f;
    }
    if (a.coords != nullptr) {
        float* c = a.coords + (size_t)i * a.coord_stride * 3;
#pragma unroll
        for (int j = 0; j < J; ++j)
            if (L.valid[j]) { c[3 * L.orig[j]] = x[j]; c[3 * L.orig[j] + 1] = y[j]; c[3 * L.orig[j] + 2] = z[j]; }
        for (int e = 3 * L.n + lane; e < 3 * a.coord_stride; e += 32) c[e] = 0.f;
    }
}

template <bool MDN>
__global__ void __launch_bounds__(TRIDSK_WARPS_PER_CTA * 32) score_kernel(const ScoreLaunch a) {
    __shared__ float sP_all[TRIDSK_WARPS_PER_CTA][6 * TRIDSK_MAX_J * 32];
    const int warp = threadIdx.x >> 5;
    const int i = blockIdx.x * TRIDSK_WARPS_PER_CTA + warp;
    if (i >= a.n_pose) return;
    const int lig = a.lig_index[i];
    switch (a.hdr[lig].J) {                 // warp-uniform
        case 1: score_one<1, MDN>(a, i, lig, sP_all[warp]); break;
        case 2: score_one<2, MDN>(a, i, lig, sP_all[warp]); break;
        case 3: score_one<3, MDN>(a, i, lig, sP_all[warp]); break;
        default: score_one<4, MDN>(a, i, lig, sP_all[warp]); break;
    }
}

cudaError_t launch_score(cudaStream_t s, const ScoreLaunch& a) {
    if (a.n_pose <= 0) return cudaSuccess;
    const int blocks = (a.n_pose + TRIDSK_WARPS_PER_CTA - 1) / TRIDSK_WARPS_PER_CTA;
    if (a.mdn.n_res > 0) score_kernel<true><<<blocks, TRIDSK_WARPS_PER_CTA * 32, 0, s>>>(a);
    else score_kernel<false><<<blocks, TRIDSK_WARPS_PER_CTA * 32, 0, s>>>(a);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ O10 test hook
__global__ void philox_debug_kernel(const unsigned int* ck, unsigned int* out) {
    const uint4 r = philox4x32_10(make_uint4(ck[0], ck[1], ck[2], ck[3]), make_uint2(ck[4], ck[5]));
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
cudaError_t launch_philox_debug(cudaStream_t s, const unsigned int* ctr_key, unsigned int* out) {
    philox_debug_kernel<<<1, 1, 0, s>>>(ctr_key, out);
    return cudaGetLastError();
}
