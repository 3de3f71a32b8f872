// mc_lane.cu -- the throughput form of the fused per-chain Monte Carlo kernel (steps a1..a8, a10): one LANE per
// chain, one CTA = up to 128 chains of ONE ligand.
//
// Why a second mapping.  With a warp per chain (mc_kernel.cu) a 30-atom ligand costs ~2,100 warp instructions per
// pose evaluation: partner coordinates and reaction forces travel by shuffles, a third of the lanes idle in every
// pair round, and the tree passes are scans.  When there are far more chains than lanes (screens: 0.5-4 M chains),
// giving every lane its own chain removes all of that: the ligand topology is warp-uniform (staged once per CTA in
// shared memory, read as broadcasts), pair constants are per-pair scalars, loops have uniform trip counts, and the
// only divergence left is the distance cut-offs.  ~450 warp instructions per evaluation for the same ligand.
//
// Shared memory per CTA: topology {ref xyz + type, fragment records, pair list grouped by first atom} + per chain,
// slot-major ([slot][chain], so lanes hit distinct banks): coordinates X[3n], forces F[max(3n, 12(T+1))] -- the
// fragment frames of the forward pass alias F, which is dead until the gather writes it -- and the current /
// proposed torsion angles.  The rigid pose, Adam moments of the rigid DoFs and the energies live in registers; the
// best pose goes straight to global memory when it improves.  No atomics anywhere: bit-reproducible.
//
// P:N = PAPER.md line N; O*/G* = DESIGN.md section 3.
#include "chain.cuh"

struct LaneTopo {
    const float4* ref;      // [n] {ref x, y, z, type bits}
    const FragRec* frag;    // [T + 1]
    const uint2* pair;      // [P] {b | hb << 8, d_vdw bits}, grouped by first atom
    const int* pstart;      // [n + 1]
    int n, T;
};

// Stage one ligand's topology into shared memory; returns the first byte after it (16-byte aligned).
__device__ __forceinline__ unsigned char* lane_stage(LaneTopo& S, unsigned char* smem, const LigHdr* __restrict__ h,
                                                     const float4* __restrict__ atom_f4, const int* __restrict__ atom_i,
                                                     const FragRec* __restrict__ frags, const uint2* __restrict__ lane_pairs,
                                                     const int* __restrict__ lane_pstart) {
    const int n = h->n, T = h->T, P = h->n_pairs, tid = threadIdx.x, nt = blockDim.x;
    float4* ref = reinterpret_cast<float4*>(smem);
    int* frag = reinterpret_cast<int*>(smem + 16 * (size_t)n);
    uint2* pair = reinterpret_cast<uint2*>(smem + 16 * (size_t)n + sizeof(FragRec) * (size_t)(T + 1));
    int* pstart = reinterpret_cast<int*>(reinterpret_cast<unsigned char*>(pair) + 8 * (size_t)P);
    for (int i = tid; i < n; i += nt) {
        const float4 f = __ldg(atom_f4 + h->atom_off + i);
        ref[i] = make_float4(f.x, f.y, f.z, __int_as_float(__ldg(atom_i + h->atom_off + i) & 0xff));
    }
    const int* fsrc = reinterpret_cast<const int*>(frags + h->frag_off);
    for (int i = tid; i < (T + 1) * (int)(sizeof(FragRec) / 4); i += nt) frag[i] = __ldg(fsrc + i);
    for (int i = tid; i < P; i += nt) pair[i] = __ldg(lane_pairs + h->lp_off + i);
    for (int i = tid; i <= n; i += nt) pstart[i] = __ldg(lane_pstart + h->ps_off + i);
    S.ref = ref; S.frag = reinterpret_cast<const FragRec*>(frag); S.pair = pair; S.pstart = pstart; S.n = n; S.T = T;
    return smem + lane_topo_bytes(n, T, P);
}

// x_a = R r_a + p for the fragment's own atoms [lo, hi)
__device__ __forceinline__ void lane_place(const LaneTopo& S, const float R[9], const float p[3], int lo, int hi,
                                           float* __restrict__ X, int C) {
    for (int a = lo; a < hi; ++a) {
        const float4 r = S.ref[a];
        float* xa = X + 3 * a * C;
        xa[0] = fmaf(R[0], r.x, fmaf(R[1], r.y, fmaf(R[2], r.z, p[0])));
        xa[C] = fmaf(R[3], r.x, fmaf(R[4], r.y, fmaf(R[5], r.z, p[1])));
        xa[2 * C] = fmaf(R[6], r.x, fmaf(R[7], r.y, fmaf(R[8], r.z, p[2])));
    }
}

// ------------------------------------------------------------------ a3..a5: one pose evaluation by one lane
// In : t[3], unit q[4] (registers), th[k*C] torsion angles (shared).
// Out: X (world coordinates), e_inter, e_intra; GRAD: F[a] = dE/dx_a.
template <bool GRAD>
__device__ __forceinline__ void lane_eval(const LaneTopo& S, const DGrid& G, const DParams& P, const float t[3],
                                          const float q[4], const float* __restrict__ th, float* __restrict__ X,
                                          float* __restrict__ F, int C, float& e_inter, float& e_intra) {
    // ---- a3 forward kinematics (O8): fragment frames F_f = F_parent o L_f in index order (parents precede children);
    // a frame is 12 slots of the (still dead) force region; every fragment places its own atoms while its frame is
    // in registers.
    {
        float R[9], p[3];
        quat_matrix(q, R);
        p[0] = t[0]; p[1] = t[1]; p[2] = t[2];
        if (S.T > 0) {
#pragma unroll
            for (int i = 0; i < 9; ++i) F[i * C] = R[i];
#pragma unroll
            for (int i = 0; i < 3; ++i) F[(9 + i) * C] = p[i];
        }
        lane_place(S, R, p, 0, S.frag[0].own_hi, X, C);
        for (int f = 1; f <= S.T; ++f) {
            const FragRec& r = S.frag[f];
            const float ux = r.ux, uy = r.uy, uz = r.uz, ox = r.ox, oy = r.oy, oz = r.oz;
            float sn, cs;
            sincosf(th[(f - 1) * C], &sn, &cs);
            const float oc = 1.f - cs;
            float Lm[9];
            Lm[0] = fmaf(oc * ux, ux, cs);        Lm[1] = fmaf(oc * ux, uy, -sn * uz);  Lm[2] = fmaf(oc * ux, uz, sn * uy);
            Lm[3] = fmaf(oc * uy, ux, sn * uz);   Lm[4] = fmaf(oc * uy, uy, cs);        Lm[5] = fmaf(oc * uy, uz, -sn * ux);
            Lm[6] = fmaf(oc * uz, ux, -sn * uy);  Lm[7] = fmaf(oc * uz, uy, sn * ux);   Lm[8] = fmaf(oc * uz, uz, cs);
            const float c0 = ox - (Lm[0] * ox + Lm[1] * oy + Lm[2] * oz);         // L_f(x) = Lm x + c
            const float c1 = oy - (Lm[3] * ox + Lm[4] * oy + Lm[5] * oz);
            const float c2 = oz - (Lm[6] * ox + Lm[7] * oy + Lm[8] * oz);
            const float* PF = F + 12 * r.parent * C;
            float PR[9], pp[3];
#pragma unroll
            for (int i = 0; i < 9; ++i) PR[i] = PF[i * C];
#pragma unroll
            for (int i = 0; i < 3; ++i) pp[i] = PF[(9 + i) * C];
#pragma unroll
            for (int rr = 0; rr < 3; ++rr) {
                R[3 * rr + 0] = PR[3 * rr] * Lm[0] + PR[3 * rr + 1] * Lm[3] + PR[3 * rr + 2] * Lm[6];
                R[3 * rr + 1] = PR[3 * rr] * Lm[1] + PR[3 * rr + 1] * Lm[4] + PR[3 * rr + 2] * Lm[7];
                R[3 * rr + 2] = PR[3 * rr] * Lm[2] + PR[3 * rr + 1] * Lm[5] + PR[3 * rr + 2] * Lm[8];
                p[rr] = PR[3 * rr] * c0 + PR[3 * rr + 1] * c1 + PR[3 * rr + 2] * c2 + pp[rr];
            }
            if (r.hi > r.own_hi) {                 // it has children: they will read this frame
                float* MF = F + 12 * f * C;
#pragma unroll
                for (int i = 0; i < 9; ++i) MF[i * C] = R[i];
#pragma unroll
                for (int i = 0; i < 3; ++i) MF[(9 + i) * C] = p[i];
            }
            lane_place(S, R, p, r.lo, r.own_hi, X, C);
        }
    }

    // ---- a4 receptor energy: two 16-byte records of the xy-packed grid per atom; GRAD: F[a] <- grid gradient
    e_inter = 0.f;
#pragma unroll 2
    for (int a = 0; a < S.n; ++a) {
        const float* xa = X + 3 * a * C;
        float gx, gy, gz;
        e_inter += grid_interp_packed<GRAD>(G, P.k_wall, __float_as_int(S.ref[a].w), xa[0], xa[C], xa[2 * C], gx, gy, gz);
        if (GRAD) {
            float* fa = F + 3 * a * C;
            fa[0] = gx; fa[C] = gy; fa[2 * C] = gz;
        }
    }

    // ---- a5 intra-ligand pairs, grouped by first atom: its force accumulates in registers, the partner's in F
    e_intra = 0.f;
    for (int a = 0; a < S.n; ++a) {
        const int pb = S.pstart[a], pe = S.pstart[a + 1];
        if (pb == pe) continue;
        const float* xa = X + 3 * a * C;
        const float ax = xa[0], ay = xa[C], az = xa[2 * C];
        float sx = 0.f, sy = 0.f, sz = 0.f;
#pragma unroll 2
        for (int i = pb; i < pe; ++i) {
            const uint2 pr = S.pair[i];
            const int b = pr.x & 0xff;
            const float* xb = X + 3 * b * C;
            const float dx = ax - xb[0], dy = ay - xb[C], dz = az - xb[2 * C];
            float s;
            e_intra += pair_energy<GRAD>(P, dx * dx + dy * dy + dz * dz, __uint_as_float(pr.y), (pr.x >> 8) & 1u, s);
            if (GRAD) {
                const float px = s * dx, py = s * dy, pz = s * dz;
                sx += px; sy += py; sz += pz;
                float* fb = F + 3 * b * C;
                fb[0] -= px; fb[C] -= py; fb[2 * C] -= pz;
            }
        }
        if (GRAD) {
            float* fa = F + 3 * a * C;
            fa[0] += sx; fa[C] += sy; fa[2 * C] += sz;
        }
    }
}

// ------------------------------------------------------------------ a6 reverse mode (O9)
// Rigid part: dE/dt = sum g_a, dE/domega = sum (x_a - t) x g_a.
__device__ __forceinline__ void lane_rigid_grad(const LaneTopo& S, const float t[3], const float* __restrict__ X,
                                                const float* __restrict__ F, int C, float g[6]) {
    float fx = 0.f, fy = 0.f, fz = 0.f, mx = 0.f, my = 0.f, mz = 0.f;
#pragma unroll 2
    for (int a = 0; a < S.n; ++a) {
        const float* xa = X + 3 * a * C;
        const float* fa = F + 3 * a * C;
        const float rx = xa[0] - t[0], ry = xa[C] - t[1], rz = xa[2 * C] - t[2];
        const float gx = fa[0], gy = fa[C], gz = fa[2 * C];
        fx += gx; fy += gy; fz += gz;
        mx += ry * gz - rz * gy; my += rz * gx - rx * gz; mz += rx * gy - ry * gx;
    }
    g[0] = fx; g[1] = fy; g[2] = fz; g[3] = mx; g[4] = my; g[5] = mz;
}
// Torsion k: dE/dtheta_k = u_k . sum_{a in subtree(k)} (x_a - x_bk) x g_a, u_k = unit(x_bk - x_ak) in the world frame;
// the subtree is the contiguous atom range [lo, hi) of the depth-first order.
__device__ __forceinline__ float lane_torsion_grad(const LaneTopo& S, int k, const float* __restrict__ X,
                                                   const float* __restrict__ F, int C) {
    const FragRec& r = S.frag[k + 1];
    const int ia = r.axis & 0xff, ib = (r.axis >> 8) & 0xff;
    const float* xb = X + 3 * ib * C;
    const float* xa = X + 3 * ia * C;
    const float ox = xb[0], oy = xb[C], oz = xb[2 * C];
    float ux = ox - xa[0], uy = oy - xa[C], uz = oz - xa[2 * C];
    const float un = rsqrtf(ux * ux + uy * uy + uz * uz);
    ux *= un; uy *= un; uz *= un;
    float mx = 0.f, my = 0.f, mz = 0.f;
#pragma unroll 2
    for (int a = r.lo; a < r.hi; ++a) {
        const float* xc = X + 3 * a * C;
        const float* fc = F + 3 * a * C;
        const float rx = xc[0] - ox, ry = xc[C] - oy, rz = xc[2 * C] - oz;
        const float gx = fc[0], gy = fc[C], gz = fc[2 * C];
        mx += ry * gz - rz * gy; my += rz * gx - rx * gz; mz += rx * gy - ry * gx;
    }
    return ux * mx + uy * my + uz * mz;
}

// ------------------------------------------------------------------ the fused MC kernel, one lane per chain
__global__ void __launch_bounds__(128) mc_lane_kernel(const McLaunch a) {
    extern __shared__ __align__(16) unsigned char lane_smem[];
    const int C = blockDim.x, tid = threadIdx.x;
    const int cpl = (a.n_chains + C - 1) / C;                 // CTAs per ligand
    const int lig = a.lig_list[blockIdx.x / cpl];
    const int chain = (blockIdx.x % cpl) * C + tid;
    LaneTopo S;
    unsigned char* after = lane_stage(S, lane_smem, a.hdr + lig, a.atom_f4, a.atom_i, a.frags, a.lane_pairs, a.lane_pstart);
    __syncthreads();
    if (chain >= a.n_chains) return;

    const DParams& P = a.P;
    const int n = S.n, T = S.T;
    float* X = reinterpret_cast<float*>(after) + tid;         // slot-major: slot i of this chain is X[i * C]
    float* F = X + 3 * n * C;
    float* THC = F + lane_fslots(n, T) * C;                   // current accepted torsions
    float* THP = THC + T * C;                                 // proposal
    float* MV = THP + T * C;                                  // torsion Adam moments {m_k, v_k} (n_refine > 1 only)
    const size_t cidx = (size_t)lig * a.n_chains + chain;
    const uint2 key = make_uint2((uint32_t)a.seed, (uint32_t)(a.seed >> 32));
    const uint32_t gchain = (uint32_t)(a.chain_base + chain);
    float* g_best = a.pose_best + cidx * a.pose_stride;

    float ct[3], cq[4], ecur, ebest;
    if (a.init_mode == 2) {                                   // resume: the best pose is already in global memory
        const float* src = a.pose_cur + cidx * a.pose_stride;
        ct[0] = src[0]; ct[1] = src[1]; ct[2] = src[2];
        cq[0] = src[3]; cq[1] = src[4]; cq[2] = src[5]; cq[3] = src[6];
        for (int k = 0; k < T; ++k) THC[k * C] = src[7 + k];
        ecur = a.e_cur[cidx]; ebest = a.e_best[cidx];
    } else {
        if (a.init_mode == 1) {
            const float* src = a.init_poses + cidx * a.pose_stride;
            ct[0] = src[0]; ct[1] = src[1]; ct[2] = src[2];
            cq[0] = src[3]; cq[1] = src[4]; cq[2] = src[5]; cq[3] = src[6];
            quat_normalise(cq);
            for (int k = 0; k < T; ++k) THC[k * C] = src[7 + k];
        } else {                                              // a1 / O11: Philox initialisation
            const uint4 r2 = philox4x32_10(make_uint4(gchain, 0u, (uint32_t)lig, 2u), key);
            const float a0 = u01(r2.x), a1 = u01(r2.y), a2 = u01(r2.z);
            const float rr = a.radius * cbrtf(a0), zz = 2.f * a1 - 1.f, sq = sqrtf(fmaxf(1.f - zz * zz, 0.f));
            float sn, cs;
            sincosf(2.f * PI_F * a2, &sn, &cs);
            ct[0] = a.centre[0] + rr * sq * cs; ct[1] = a.centre[1] + rr * sq * sn; ct[2] = a.centre[2] + rr * zz;
            const uint4 r3 = philox4x32_10(make_uint4(gchain, 0u, (uint32_t)lig, 3u), key);
            const float b0 = u01(r3.x), b1 = u01(r3.y), b2 = u01(r3.z);
            const float s1 = sqrtf(1.f - b0), s2 = sqrtf(b0);
            float sn1, cs1, sn2, cs2;
            sincosf(2.f * PI_F * b1, &sn1, &cs1);
            sincosf(2.f * PI_F * b2, &sn2, &cs2);
            cq[0] = s2 * cs2; cq[1] = s1 * sn1; cq[2] = s1 * cs1; cq[3] = s2 * sn2;
            quat_normalise(cq);
            for (int k0 = 0; k0 < T; k0 += 4) {               // torsion k takes element k % 4 of block 4 + k / 4
                const uint4 r = philox4x32_10(make_uint4(gchain, 0u, (uint32_t)lig, 4u + (uint32_t)(k0 >> 2)), key);
                const uint32_t w[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    if (k0 + i < T) THC[(k0 + i) * C] = PI_F * (2.f * u01(w[i]) - 1.f);
            }
        }
        float ei, ea;
        lane_eval<false>(S, a.grid, P, ct, cq, THC, X, F, C, ei, ea);
        ecur = ei + ea;
        ebest = ecur;
        g_best[0] = ct[0]; g_best[1] = ct[1]; g_best[2] = ct[2];
        g_best[3] = cq[0]; g_best[4] = cq[1]; g_best[5] = cq[2]; g_best[6] = cq[3];
        for (int k = 0; k < T; ++k) g_best[7 + k] = THC[k * C];
        for (int e = 7 + T; e < a.pose_stride; ++e) g_best[e] = 0.f;
    }

    for (int s = 0; s < a.n_steps; ++s) {
        const uint32_t step = (uint32_t)(a.first_step + s);
        const uint4 r = philox4x32_10(make_uint4(gchain, step, (uint32_t)lig, 0u), key);      // O10: perturbation block
        const float u0 = u01(r.x), u1 = u01(r.y), u2 = u01(r.z), u3 = u01(r.w);

        // a2 / O12: perturb one entity of {translation, rotation, torsion k}
        float pt[3] = {ct[0], ct[1], ct[2]}, pq[4] = {cq[0], cq[1], cq[2], cq[3]};
        for (int k = 0; k < T; ++k) THP[k * C] = THC[k * C];
        const int entity = min((int)(u0 * (float)(T + 2)), T + 1);
        if (entity == 0) {
            pt[0] = fminf(fmaxf(pt[0] + P.pert_trans * (2.f * u1 - 1.f), a.box_min[0]), a.box_max[0]);
            pt[1] = fminf(fmaxf(pt[1] + P.pert_trans * (2.f * u2 - 1.f), a.box_min[1]), a.box_max[1]);
            pt[2] = fminf(fmaxf(pt[2] + P.pert_trans * (2.f * u3 - 1.f), a.box_min[2]), a.box_max[2]);
        } else if (entity == 1) {
            quat_rotate_by(pq, P.pert_rot * (2.f * u1 - 1.f), P.pert_rot * (2.f * u2 - 1.f), P.pert_rot * (2.f * u3 - 1.f));
        } else {
            THP[(entity - 2) * C] = PI_F * (2.f * u1 - 1.f);
        }

        // a3..a7: n_refine Adam steps on the 6+T tangent components (moments reset every MC step, G12)
        float m[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, v[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        float b1p = 1.f, b2p = 1.f;
        for (int rf = 0; rf < P.n_refine; ++rf) {
            float ei, ea;
            lane_eval<true>(S, a.grid, P, pt, pq, THP, X, F, C, ei, ea);
            b1p *= P.adam_b1; b2p *= P.adam_b2;
            const float c1 = 1.f / (1.f - b1p), c2 = 1.f / (1.f - b2p);
            float g[6];
            lane_rigid_grad(S, pt, X, F, C, g);
            for (int k = 0; k < T; ++k) {                     // torsion gradients are consumed as they are produced
                const float gk = lane_torsion_grad(S, k, X, F, C);
                float mk = 0.f, vk = 0.f;
                if (rf > 0) { mk = MV[2 * k * C]; vk = MV[(2 * k + 1) * C]; }
                mk = P.adam_b1 * mk + (1.f - P.adam_b1) * gk;
                vk = P.adam_b2 * vk + (1.f - P.adam_b2) * gk * gk;
                if (rf + 1 < P.n_refine) { MV[2 * k * C] = mk; MV[(2 * k + 1) * C] = vk; }
                float th = THP[k * C] - P.lr * (mk * c1) / (sqrtf(vk * c2) + P.adam_eps);
                if (th >= PI_F) th -= 2.f * PI_F;
                if (th < -PI_F) th += 2.f * PI_F;
                THP[k * C] = th;
            }
            float dl[6];
#pragma unroll
            for (int i = 0; i < 6; ++i) {
                m[i] = P.adam_b1 * m[i] + (1.f - P.adam_b1) * g[i];
                v[i] = P.adam_b2 * v[i] + (1.f - P.adam_b2) * g[i] * g[i];
                dl[i] = -P.lr * (m[i] * c1) / (sqrtf(v[i] * c2) + P.adam_eps);
            }
            pt[0] = fminf(fmaxf(pt[0] + dl[0], a.box_min[0]), a.box_max[0]);
            pt[1] = fminf(fmaxf(pt[1] + dl[1], a.box_min[1]), a.box_max[1]);
            pt[2] = fminf(fmaxf(pt[2] + dl[2], a.box_min[2]), a.box_max[2]);
            quat_rotate_by(pq, dl[3], dl[4], dl[5]);
        }

        // a8: energy of the refined proposal, Metropolis, best tracking
        float ei, ea;
        lane_eval<false>(S, a.grid, P, pt, pq, THP, X, F, C, ei, ea);
        const float enew = ei + ea;
        const uint4 rm = philox4x32_10(make_uint4(gchain, step, (uint32_t)lig, 1u), key);     // Metropolis block
        const float um = u01(rm.x);
        const bool accept = isfinite(enew) && (um < expf(-P.beta * (enew - ecur)));
        if (a.trace != nullptr) {
            tridsk_trace_rec rec;
            rec.e_prop = enew; rec.e_cur = ecur; rec.u = um; rec.flags = (accept ? 1 : 0) | (entity << 8);
            a.trace[cidx * a.trace_stride + a.trace_off + s] = rec;
        }
        if (accept) {
#pragma unroll
            for (int i = 0; i < 3; ++i) ct[i] = pt[i];
#pragma unroll
            for (int i = 0; i < 4; ++i) cq[i] = pq[i];
            for (int k = 0; k < T; ++k) THC[k * C] = THP[k * C];
            ecur = enew;
            if (enew < ebest) {
                ebest = enew;
                g_best[0] = pt[0]; g_best[1] = pt[1]; g_best[2] = pt[2];
                g_best[3] = pq[0]; g_best[4] = pq[1]; g_best[5] = pq[2]; g_best[6] = pq[3];
                for (int k = 0; k < T; ++k) g_best[7 + k] = THP[k * C];
            }
        }
    }

    float* dst = a.pose_cur + cidx * a.pose_stride;
    dst[0] = ct[0]; dst[1] = ct[1]; dst[2] = ct[2];
    dst[3] = cq[0]; dst[4] = cq[1]; dst[5] = cq[2]; dst[6] = cq[3];
    for (int k = 0; k < T; ++k) dst[7 + k] = THC[k * C];
    for (int e = 7 + T; e < a.pose_stride; ++e) dst[e] = 0.f;
    a.e_cur[cidx] = ecur; a.e_best[cidx] = ebest;
}

static bool g_lane_prepared = false;
cudaError_t mc_lane_prepare(size_t max_smem_bytes);

cudaError_t launch_mc_lane(cudaStream_t s, const McLaunch& a, int chains_per_cta, size_t smem_bytes) {
    const int cpl = (a.n_chains + chains_per_cta - 1) / chains_per_cta;
    const long long blocks = (long long)a.n_list * cpl;
    if (blocks <= 0) return cudaSuccess;
    if (blocks > 0x7fffffffLL || chains_per_cta < 32 || chains_per_cta > 128 || (chains_per_cta & 31)) return cudaErrorInvalidValue;
    cudaError_t e = mc_lane_prepare(TRIDSK_SMEM_MAX_CTA);
    if (e != cudaSuccess) return e;
    mc_lane_kernel<<<(unsigned)blocks, chains_per_cta, smem_bytes, s>>>(a);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ tridsk_score_grad, lane form: one lane per pose
// One 32-thread CTA takes up to 32 poses of one ligand (the host groups poses by ligand: seg_*, perm).
__global__ void __launch_bounds__(32) score_lane_kernel(const ScoreLaunch a) {
    extern __shared__ __align__(16) unsigned char lane_smem[];
    const int C = 32, tid = threadIdx.x;
    const int lig = a.seg_lig[blockIdx.x];
    const LigHdr* h = a.hdr + lig;
    LaneTopo S;
    unsigned char* after = lane_stage(S, lane_smem, h, a.atom_f4, a.atom_i, a.frags, a.lane_pairs, a.lane_pstart);
    __syncthreads();
    if (tid >= a.seg_cnt[blockIdx.x]) return;
    const int i = a.perm[a.seg_start[blockIdx.x] + tid];
    const int n = S.n, T = S.T;
    float* X = reinterpret_cast<float*>(after) + tid;
    float* F = X + 3 * n * C;
    float* TH = F + lane_fslots(n, T) * C;
    const float* src = a.poses + (size_t)i * a.pose_stride;
    float t[3] = {src[0], src[1], src[2]}, q[4] = {src[3], src[4], src[5], src[6]};
    quat_normalise(q);
    for (int k = 0; k < T; ++k) TH[k * C] = src[7 + k];
    float ei, ea;
    if (a.grad != nullptr) lane_eval<true>(S, a.grid, a.P, t, q, TH, X, F, C, ei, ea);
    else lane_eval<false>(S, a.grid, a.P, t, q, TH, X, F, C, ei, ea);
    a.energy[3 * (size_t)i] = ei + ea; a.energy[3 * (size_t)i + 1] = ei; a.energy[3 * (size_t)i + 2] = ea;
    if (a.grad != nullptr) {
        float* g = a.grad + (size_t)i * a.grad_stride;
        float gr[6];
        lane_rigid_grad(S, t, X, F, C, gr);
#pragma unroll
        for (int c = 0; c < 6; ++c) g[c] = gr[c];
        for (int k = 0; k < T; ++k) g[6 + k] = lane_torsion_grad(S, k, X, F, C);
        for (int e = 6 + T; e < a.grad_stride; ++e) g[e] = 0.f;
    }
    if (a.coords != nullptr) {
        float* c = a.coords + (size_t)i * a.coord_stride * 3;
        for (int p = 0; p < n; ++p) {
            const int orig = (__ldg(a.atom_i + h->atom_off + p) >> 16) & 0xff;
            c[3 * orig] = X[3 * p * C]; c[3 * orig + 1] = X[(3 * p + 1) * C]; c[3 * orig + 2] = X[(3 * p + 2) * C];
        }
        for (int e = 3 * n; e < 3 * a.coord_stride; ++e) c[e] = 0.f;
    }
}

cudaError_t mc_lane_prepare(size_t max_smem_bytes) {
    if (g_lane_prepared) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(mc_lane_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_smem_bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(score_lane_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_smem_bytes);
    if (e == cudaSuccess) g_lane_prepared = true;
    return e;
}

cudaError_t launch_score_lane(cudaStream_t s, const ScoreLaunch& a, int n_seg, size_t smem_bytes) {
    if (n_seg <= 0) return cudaSuccess;
    cudaError_t e = mc_lane_prepare(TRIDSK_SMEM_MAX_CTA);
    if (e != cudaSuccess) return e;
    score_lane_kernel<<<n_seg, 32, smem_bytes, s>>>(a);
    return cudaGetLastError();
}
