// score_direct.cu -- tridsk_score_direct: pose energy and gradient with the receptor term taken
// the paper's own way (P:103-125, P:353 item 4) -- direct sums over the receptor atoms within the cut-off, no grid, no
// interpolation, no wall.  It is what the grid tabulates (O3), so the difference to tridsk_score_grad is the
// interpolation error of the hot path's receptor term; it is a measuring tool, not part of the MC loop.
//
// One CTA (128 threads) per pose.  Forward kinematics as in topk_cluster_kernel (one thread per fragment composes its
// frame from the root down, O8); receptor term: a warp per ligand atom, lanes stride over the receptor atoms, fixed-order
// shuffle reduction; intra term: the CTA format's row form (a warp per atom walks the atom's partners); reverse pass (O9):
// one thread per fragment sums its subtree's atom range.  No atomics: bit-reproducible.
#include "chain.cuh"

#define SD_THREADS 128

struct DirectLaunch {
    const LigHdr* hdr;
    const float4* atom_f4; const int* atom_i; const LaneFrag* lane_frags;
    const int* cta_rows; const uint2* cta_recs;
    const float4* rec;            // {x, y, z, type bits}
    int n_rec;
    const float* radius;          // [n_types]
    const unsigned char* role;    // [n_types]
    DParams P;
    const int* lig_index; const float* poses; int n_pose, pose_stride;
    float* energy; float* grad; int grad_stride;
    int max_atoms;
};

__global__ void __launch_bounds__(SD_THREADS) score_direct_kernel(const DirectLaunch a) {
    extern __shared__ __align__(16) float sd_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, i = blockIdx.x;
    const int lig = a.lig_index[i];
    const LigHdr h = a.hdr[lig];
    const int n = h.n, T = h.T;
    float* X = sd_smem;                       // [n][3]
    float* G = X + 3 * a.max_atoms;           // [n][3] dE/dx_a
    float* EA = G + 3 * a.max_atoms;          // [n][2] per-atom receptor / intra energy
    const float4* ref = a.atom_f4 + h.atom_off;
    const LaneFrag* frag = a.lane_frags + h.frag_off;
    const float* pose = a.poses + (size_t)i * a.pose_stride;
    const DParams& P = a.P;

    // a3 / O8: thread g composes the frame of fragment g along its ancestors and places the fragment's own atoms
    if (tid <= T) {
        int path[TRIDSK_MAX_TORSIONS + 1], np_ = 0;
        for (int g = tid; g > 0; g = frag[g].parent) path[np_++] = g;
        float q[4] = {pose[3], pose[4], pose[5], pose[6]};
        quat_normalise(q);
        float R[9], p[3] = {pose[0], pose[1], pose[2]};
        quat_matrix(q, R);
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
            for (int k2 = 0; k2 < 9; ++k2) R[k2] = Rn[k2];
#pragma unroll
            for (int k2 = 0; k2 < 3; ++k2) p[k2] = pn[k2];
        }
        const LaneFrag me = frag[tid];
        for (int at = me.lo; at < me.own_hi; ++at) {
            const float4 r = ref[at];
            X[3 * at] = R[0] * r.x + R[1] * r.y + R[2] * r.z + p[0];
            X[3 * at + 1] = R[3] * r.x + R[4] * r.y + R[5] * r.z + p[1];
            X[3 * at + 2] = R[6] * r.x + R[7] * r.y + R[8] * r.z + p[2];
        }
    }
    __syncthreads();

    // per ligand atom (a warp each): receptor term over all receptor atoms, intra term over the atom's row
    const int* rows = a.cta_rows + h.cta_row_off;
    const uint2* recs = a.cta_recs + h.cta_rec_off;
    for (int at = warp; at < n; at += SD_THREADS / 32) {
        const float x = X[3 * at], y = X[3 * at + 1], z = X[3 * at + 2];
        const int ta = a.atom_i[h.atom_off + at] & 0xff;
        const float ra = a.radius[ta];
        const unsigned char ro = a.role[ta];
        float er = 0.f, ei = 0.f, gx = 0.f, gy = 0.f, gz = 0.f;
        for (int r = lane; r < a.n_rec; r += 32) {
            const float4 q = __ldg(a.rec + r);
            const int s = __float_as_int(q.w);
            if (s < 0) continue;
            const float dx = x - q.x, dy = y - q.y, dz = z - q.z;
            const unsigned char rs = a.role[s];
            const bool hb = ((rs & 1) && (ro & 2)) || ((rs & 2) && (ro & 1));
            float sod;
            er += pair_energy<true>(P, dx * dx + dy * dy + dz * dz, a.radius[s] + ra, hb, sod);
            gx = fmaf(sod, dx, gx); gy = fmaf(sod, dy, gy); gz = fmaf(sod, dz, gz);
        }
        for (int k = rows[at] + lane; k < rows[at + 1]; k += 32) {
            const uint2 rec = recs[k];
            const int b = (int)(rec.x & 0xffu);
            const float dx = x - X[3 * b], dy = y - X[3 * b + 1], dz = z - X[3 * b + 2];
            float sod;
            ei += pair_energy<true>(P, dx * dx + dy * dy + dz * dz, __uint_as_float(rec.y), (rec.x >> 8) & 1u, sod);
            gx = fmaf(sod, dx, gx); gy = fmaf(sod, dy, gy); gz = fmaf(sod, dz, gz);
        }
        er = warp_sum(er); ei = warp_sum(ei); gx = warp_sum(gx); gy = warp_sum(gy); gz = warp_sum(gz);
        if (lane == 0) { G[3 * at] = gx; G[3 * at + 1] = gy; G[3 * at + 2] = gz; EA[2 * at] = er; EA[2 * at + 1] = 0.5f * ei; }
    }
    __syncthreads();

    if (tid == 0) {
        float er = 0.f, ei = 0.f;
        for (int at = 0; at < n; ++at) { er += EA[2 * at]; ei += EA[2 * at + 1]; }
        a.energy[3 * (size_t)i] = er + ei; a.energy[3 * (size_t)i + 1] = er; a.energy[3 * (size_t)i + 2] = ei;
    }
    if (a.grad == nullptr) return;
    // a6 / O9: thread g sums the atom range of its subtree
    float* gr = a.grad + (size_t)i * a.grad_stride;
    if (tid <= T) {
        int e = tid + 1;
        while (e <= T && frag[e].depth > frag[tid].depth) ++e;
        const int lo = frag[tid].lo, hi = frag[e - 1].own_hi;
        const LaneFrag me = frag[tid];
        const int ia = me.axis & 0xff, ib = (me.axis >> 8) & 0xff;
        // reference point: t for the rigid part (fragment 0), the axis atom b for a torsion
        const float px = tid == 0 ? pose[0] : X[3 * ib], py = tid == 0 ? pose[1] : X[3 * ib + 1], pz = tid == 0 ? pose[2] : X[3 * ib + 2];
        float F[3] = {0.f, 0.f, 0.f}, M[3] = {0.f, 0.f, 0.f};
        for (int at = lo; at < hi; ++at) {
            const float rx = X[3 * at] - px, ry = X[3 * at + 1] - py, rz = X[3 * at + 2] - pz;
            const float fx = G[3 * at], fy = G[3 * at + 1], fz = G[3 * at + 2];
            F[0] += fx; F[1] += fy; F[2] += fz;
            M[0] += ry * fz - rz * fy; M[1] += rz * fx - rx * fz; M[2] += rx * fy - ry * fx;
        }
        if (tid == 0) {
            gr[0] = F[0]; gr[1] = F[1]; gr[2] = F[2]; gr[3] = M[0]; gr[4] = M[1]; gr[5] = M[2];
        } else {
            float ux = X[3 * ib] - X[3 * ia], uy = X[3 * ib + 1] - X[3 * ia + 1], uz = X[3 * ib + 2] - X[3 * ia + 2];
            const float un = rsqrtf(ux * ux + uy * uy + uz * uz);
            gr[6 + me.tor] = (ux * M[0] + uy * M[1] + uz * M[2]) * un;
        }
    }
    for (int e = 6 + T + tid; e < a.grad_stride; e += SD_THREADS) gr[e] = 0.f;
}

cudaError_t launch_score_direct(cudaStream_t s, const LigHdr* hdr, const float4* atom_f4, const int* atom_i, const LaneFrag* lane_frags,
                                const int* cta_rows, const uint2* cta_recs, const float4* rec, int n_rec, const float* radius,
                                const unsigned char* role, const DParams& P, const int* lig_index, const float* poses, int n_pose,
                                int pose_stride, float* energy, float* grad, int grad_stride, int max_atoms) {
    if (n_pose <= 0) return cudaSuccess;
    DirectLaunch a;
    a.hdr = hdr; a.atom_f4 = atom_f4; a.atom_i = atom_i; a.lane_frags = lane_frags; a.cta_rows = cta_rows; a.cta_recs = cta_recs;
    a.rec = rec; a.n_rec = n_rec; a.radius = radius; a.role = role; a.P = P;
    a.lig_index = lig_index; a.poses = poses; a.n_pose = n_pose; a.pose_stride = pose_stride;
    a.energy = energy; a.grad = grad; a.grad_stride = grad_stride; a.max_atoms = max_atoms;
    const size_t smem = sizeof(float) * 8 * (size_t)max_atoms;
    score_direct_kernel<<<n_pose, SD_THREADS, smem, s>>>(a);
    return cudaGetLastError();
}
