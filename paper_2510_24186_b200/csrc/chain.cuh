// chain.cuh -- warp-cooperative device functions of the fused per-chain kernel (hot-path steps a2..a8).
//
// One warp owns one chain (BASELINE.json north_star: "one warp or CTA per chain").  Lane l owns
//   * atoms a = j*S + l (j < J "stripes", internal depth-first order): reference and world coordinates, forces;
//   * rigid fragment f = l (0 = root, k+1 = child of torsion k): its torsion angle and its world frame.
// Everything lives in registers and moves by warp shuffles; the only shared memory is a per-warp prefix-sum
// scratch used by the reverse-mode pass.  No atomics: results are bit-reproducible run to run.
//
// P:N = PAPER.md line N; O*/G* = DESIGN.md section 3.
#pragma once
#include "internal.h"
#include "mdn.cuh"

#define FULL_MASK 0xffffffffu
#define PI_F 3.14159265358979323846f

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL_MASK, v, o);
    return v;
}

// ------------------------------------------------------------------ O10: Philox4x32-10 (counter-based RNG)
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}
// u = ((r >> 9) + 0.5) 2^-23: in (0,1), exact in fp32
__device__ __forceinline__ float u01(uint32_t r) { return ((float)(r >> 9) + 0.5f) * (1.0f / 8388608.0f); }

// ------------------------------------------------------------------ small quaternion helpers (Hamilton, scalar first)
__device__ __forceinline__ void quat_normalise(float q[4]) {
    const float n = rsqrtf(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    q[0] *= n; q[1] *= n; q[2] *= n; q[3] *= n;
}
__device__ __forceinline__ void quat_matrix(const float q[4], float R[9]) {
    const float w = q[0], x = q[1], y = q[2], z = q[3];
    R[0] = 1.f - 2.f * (y * y + z * z); R[1] = 2.f * (x * y - w * z);       R[2] = 2.f * (x * z + w * y);
    R[3] = 2.f * (x * y + w * z);       R[4] = 1.f - 2.f * (x * x + z * z); R[5] = 2.f * (y * z - w * x);
    R[6] = 2.f * (x * z - w * y);       R[7] = 2.f * (y * z + w * x);       R[8] = 1.f - 2.f * (x * x + y * y);
}
// q <- normalise(exp_q(v) (x) q): left-multiply by the rotation vector v (world frame)
__device__ __forceinline__ void quat_rotate_by(float q[4], float vx, float vy, float vz) {
    const float a2 = vx * vx + vy * vy + vz * vz;
    float dw, s;
    if (a2 < 1e-16f) { dw = 1.f; s = 0.5f; }
    else {
        const float ainv = rsqrtf(a2), a = a2 * ainv;
        float sn, cs;
        __sincosf(0.5f * a, &sn, &cs);                // |a| is a fraction of a radian: abs error < 5e-7, and q is renormalised
        dw = cs; s = sn * ainv;
    }
    const float dx = s * vx, dy = s * vy, dz = s * vz;
    float r[4];
    r[0] = dw * q[0] - dx * q[1] - dy * q[2] - dz * q[3];
    r[1] = dw * q[1] + dx * q[0] + dy * q[3] - dz * q[2];
    r[2] = dw * q[2] - dx * q[3] + dy * q[0] + dz * q[1];
    r[3] = dw * q[3] + dx * q[2] - dy * q[1] + dz * q[0];
    quat_normalise(r);
    q[0] = r[0]; q[1] = r[1]; q[2] = r[2]; q[3] = r[3];
}

// ------------------------------------------------------------------ pair-function constants (lane and CTA kernels)
// Constants of the pair function in the form the inner loop wants them.
struct PairK {
    float nk2;              // -log2(e) / (2 sigma^2) of the long-range Gaussian
    float dmax;             // long-range cut-off
    float kappa;            // gradient scale: dE/dx_a = kappa * sum s (x_a - x_b),  kappa = -2 w_long / log2(e)
    float mu;               // long-range mu: the clash distance of a plain pair is c - mu
    float hb_dclash;        // clash distance of a donor/acceptor pair
    float kc;               // clash gradient in kappa units: w_clash / kappa
    float inv_floor;        // 1 / d_floor
    float kh;               // hydrogen-bond gradient in kappa units: 2 w_hbond / (2 sigma_hb^2) / kappa
    float w_long, w_clash_ln2, w_hbond, hb_dmax, hb_mu, hb_nk2;
    float neg_mu, inv_kappa, nkc;   // nkc = -kc
};
__device__ __forceinline__ PairK make_pairk(const DParams& P) {
    PairK K;
    const float L2E = 1.4426950408889634f;
    // kappa units absorb w_long; with w_long = 0 (an ablation of the term) the unit is 1 and the Gaussian is cut off at 0
    const bool has_long = P.w_long != 0.f;
    K.nk2 = -P.long_inv_two_sigma2 * L2E; K.dmax = has_long ? P.long_dmax : 0.f;
    K.kappa = has_long ? -2.f * P.w_long / L2E : 1.f;
    K.mu = P.long_mu; K.hb_dclash = P.hb_dclash;
    K.kc = P.w_clash / K.kappa; K.inv_floor = 1.f / P.d_floor;
    K.kh = 2.f * P.w_hbond * P.hb_inv_two_sigma2 / K.kappa;
    K.w_long = P.w_long; K.w_clash_ln2 = P.w_clash * 0.6931471805599453f; K.w_hbond = P.w_hbond;
    K.hb_dmax = P.hb_dmax; K.hb_mu = P.hb_mu; K.hb_nk2 = -P.hb_inv_two_sigma2 * L2E;
    K.neg_mu = -P.long_mu; K.inv_kappa = 1.f / K.kappa; K.nkc = -K.kc;
    return K;
}
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float lg2_approx(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sqrt_approx(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_approx(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// ------------------------------------------------------------------ per-chain view of one ligand, in registers
template <int J>
struct Lig {
    int n, T, S, max_depth;
    float rx[J], ry[J], rz[J], rad[J];     // reference conformer + vdW radius of this lane's atoms
    int typ[J], frg[J], orig[J];
    bool valid[J];
    float ux, uy, uz, ox, oy, oz;          // this lane's fragment: torsion axis (unit) and axis point, reference frame
    int parent, depth, lo, hi;             // parent fragment, depth, subtree atom range [lo, hi)
    const PairRound* rounds;
    int tile_off[J * (J + 1) / 2 + 1];
};

template <int J>
__device__ __forceinline__ void load_lig(Lig<J>& L, const LigHdr* __restrict__ hdrs, const float4* __restrict__ atom_f4,
                                         const int* __restrict__ atom_i, const FragRec* __restrict__ frags,
                                         const PairRound* __restrict__ rounds, int lig) {
    const int lane = threadIdx.x & 31;
    const LigHdr* h = hdrs + lig;
    L.n = h->n; L.T = h->T; L.S = h->S; L.max_depth = h->max_depth;
    L.rounds = rounds + h->round_off;
#pragma unroll
    for (int t = 0; t <= J * (J + 1) / 2; ++t) L.tile_off[t] = h->tile_off[t];
    const int ao = h->atom_off;
#pragma unroll
    for (int j = 0; j < J; ++j) {
        const int a = j * L.S + lane;
        L.valid[j] = (lane < L.S) && (a < L.n);
        float4 f = make_float4(0.f, 0.f, 0.f, 1.f);
        int w = 0;
        if (L.valid[j]) { f = __ldg(atom_f4 + ao + a); w = __ldg(atom_i + ao + a); }
        L.rx[j] = f.x; L.ry[j] = f.y; L.rz[j] = f.z; L.rad[j] = f.w;
        L.typ[j] = w & 0xff; L.frg[j] = (w >> 8) & 0xff; L.orig[j] = (w >> 16) & 0xff;
    }
    L.ux = 1.f; L.uy = 0.f; L.uz = 0.f; L.ox = 0.f; L.oy = 0.f; L.oz = 0.f;
    L.parent = 0; L.depth = 0; L.lo = 0; L.hi = 0;
    if (lane <= L.T) {
        const FragRec* fr = frags + h->frag_off + lane;
        const float4 a = __ldg(reinterpret_cast<const float4*>(fr));
        const float4 b = __ldg(reinterpret_cast<const float4*>(fr) + 1);
        const int4 c = __ldg(reinterpret_cast<const int4*>(fr) + 2);
        L.ux = a.x; L.uy = a.y; L.uz = a.z; L.ox = a.w; L.oy = b.x; L.oz = b.y;
        L.parent = c.x < 0 ? 0 : c.x; L.depth = c.x < 0 ? 0 : c.y; L.lo = c.z; L.hi = c.w;
    }
}

// ------------------------------------------------------------------ a4 / O5: trilinear receptor energy of one atom
// Value and analytic gradient of the trilinear interpolant of plane `type` at (x,y,z), plus the
// out-of-grid quadratic wall (G8).  8 explicit fp32 corner loads (texture filtering's 9-bit weights
// would break the 1e-4 tolerance).
template <bool GRAD>
__device__ __forceinline__ float grid_interp(const DGrid& G, float k_wall, int type, float x, float y, float z,
                                             float& gx, float& gy, float& gz) {
    const float ux = (x - G.ox) * G.inv_h, uy = (y - G.oy) * G.inv_h, uz = (z - G.oz) * G.inv_h;
    const float cx = fminf(fmaxf(ux, 0.f), (float)(G.nx - 1));
    const float cy = fminf(fmaxf(uy, 0.f), (float)(G.ny - 1));
    const float cz = fminf(fmaxf(uz, 0.f), (float)(G.nz - 1));
    const int ix = min((int)cx, G.nx - 2), iy = min((int)cy, G.ny - 2), iz = min((int)cz, G.nz - 2);
    const float fx = cx - (float)ix, fy = cy - (float)iy, fz = cz - (float)iz;
    const float* p = G.g + (size_t)type * G.plane + ((size_t)iz * G.ny + iy) * G.nx + ix;
    const int sy = G.nx, sz = G.nx * G.ny;
    const float v000 = __ldg(p), v001 = __ldg(p + 1), v010 = __ldg(p + sy), v011 = __ldg(p + sy + 1);
    const float v100 = __ldg(p + sz), v101 = __ldg(p + sz + 1), v110 = __ldg(p + sz + sy), v111 = __ldg(p + sz + sy + 1);
    const float d00 = v001 - v000, d01 = v011 - v010, d10 = v101 - v100, d11 = v111 - v110;   // x differences
    const float a00 = fmaf(fx, d00, v000), a01 = fmaf(fx, d01, v010), a10 = fmaf(fx, d10, v100), a11 = fmaf(fx, d11, v110);
    const float e0 = a01 - a00, e1 = a11 - a10;                                               // y differences
    const float b0 = fmaf(fy, e0, a00), b1 = fmaf(fy, e1, a10);
    float e = fmaf(fz, b1 - b0, b0);
    const bool clx = (cx != ux), cly = (cy != uy), clz = (cz != uz);
    float wx = 0.f, wy = 0.f, wz = 0.f;
    if (clx | cly | clz) {                       // rare: atom outside the grid
        wx = clx ? x - (G.ox + cx * G.h) : 0.f;
        wy = cly ? y - (G.oy + cy * G.h) : 0.f;
        wz = clz ? z - (G.oz + cz * G.h) : 0.f;
        e += k_wall * (wx * wx + wy * wy + wz * wz);
    }
    if (GRAD) {
        const float dx0 = fmaf(fy, d01 - d00, d00), dx1 = fmaf(fy, d11 - d10, d10);
        gx = (clx ? 0.f : fmaf(fz, dx1 - dx0, dx0) * G.inv_h) + 2.f * k_wall * wx;
        gy = (cly ? 0.f : fmaf(fz, e1 - e0, e0) * G.inv_h) + 2.f * k_wall * wy;
        gz = (clz ? 0.f : (b1 - b0) * G.inv_h) + 2.f * k_wall * wz;
    }
    return e;
}

// The same interpolant read from the cell-packed copy of the grid (DGrid::gp): the 8 corners of a cell are one
// aligned 32-byte record (the quads of z and z+1), i.e. one sector per atom instead of 8 loads over 4 lines.
// Arithmetic and operation order are those of grid_interp, so both give bit-identical results.
template <bool GRAD>
__device__ __forceinline__ float grid_interp_packed(const DGrid& G, float k_wall, int type, float x, float y, float z,
                                                    float& gx, float& gy, float& gz) {
    const float ux = (x - G.ox) * G.inv_h, uy = (y - G.oy) * G.inv_h, uz = (z - G.oz) * G.inv_h;
    const float cx = fminf(fmaxf(ux, 0.f), (float)(G.nx - 1));
    const float cy = fminf(fmaxf(uy, 0.f), (float)(G.ny - 1));
    const float cz = fminf(fmaxf(uz, 0.f), (float)(G.nz - 1));
    const int ix = min((int)cx, G.nx - 2), iy = min((int)cy, G.ny - 2), iz = min((int)cz, G.nz - 2);
    const float fx = cx - (float)ix, fy = cy - (float)iy, fz = cz - (float)iz;
    const float4* p = G.gp + 2 * ((size_t)type * G.plane + ((size_t)iz * G.ny + iy) * G.nx + ix);
    const float4 lo = __ldg(p), hi = __ldg(p + 1);
    const float v000 = lo.x, v001 = lo.y, v010 = lo.z, v011 = lo.w, v100 = hi.x, v101 = hi.y, v110 = hi.z, v111 = hi.w;
    const float d00 = v001 - v000, d01 = v011 - v010, d10 = v101 - v100, d11 = v111 - v110;
    const float a00 = fmaf(fx, d00, v000), a01 = fmaf(fx, d01, v010), a10 = fmaf(fx, d10, v100), a11 = fmaf(fx, d11, v110);
    const float e0 = a01 - a00, e1 = a11 - a10;
    const float b0 = fmaf(fy, e0, a00), b1 = fmaf(fy, e1, a10);
    float e = fmaf(fz, b1 - b0, b0);
    const bool clx = (cx != ux), cly = (cy != uy), clz = (cz != uz);
    float wx = 0.f, wy = 0.f, wz = 0.f;
    if (clx | cly | clz) {
        wx = clx ? x - (G.ox + cx * G.h) : 0.f;
        wy = cly ? y - (G.oy + cy * G.h) : 0.f;
        wz = clz ? z - (G.oz + cz * G.h) : 0.f;
        e += k_wall * (wx * wx + wy * wy + wz * wz);
    }
    if (GRAD) {
        const float dx0 = fmaf(fy, d01 - d00, d00), dx1 = fmaf(fy, d11 - d10, d10);
        gx = (clx ? 0.f : fmaf(fz, dx1 - dx0, dx0) * G.inv_h) + 2.f * k_wall * wx;
        gy = (cly ? 0.f : fmaf(fz, e1 - e0, e0) * G.inv_h) + 2.f * k_wall * wy;
        gz = (clz ? 0.f : (b1 - b0) * G.inv_h) + 2.f * k_wall * wz;
    }
    return e;
}

// The same interpolant in two halves, so that a caller can issue the two 16-byte loads early and blend late (the CTA
// kernel hides the L2 latency behind its pair loop).  Arithmetic and operation order are those of grid_interp.
struct GridCell {
    const float4* p;
    float fx, fy, fz, wx, wy, wz;
    bool clx, cly, clz;
};
__device__ __forceinline__ GridCell grid_locate(const DGrid& G, int type, float x, float y, float z) {
    GridCell c;
    const float ux = (x - G.ox) * G.inv_h, uy = (y - G.oy) * G.inv_h, uz = (z - G.oz) * G.inv_h;
    const float cx = fminf(fmaxf(ux, 0.f), (float)(G.nx - 1));
    const float cy = fminf(fmaxf(uy, 0.f), (float)(G.ny - 1));
    const float cz = fminf(fmaxf(uz, 0.f), (float)(G.nz - 1));
    const int ix = min((int)cx, G.nx - 2), iy = min((int)cy, G.ny - 2), iz = min((int)cz, G.nz - 2);
    c.fx = cx - (float)ix; c.fy = cy - (float)iy; c.fz = cz - (float)iz;
    c.p = G.gp + 2 * ((size_t)type * G.plane + ((size_t)iz * G.ny + iy) * G.nx + ix);
    c.clx = (cx != ux); c.cly = (cy != uy); c.clz = (cz != uz);
    c.wx = c.clx ? x - (G.ox + cx * G.h) : 0.f;
    c.wy = c.cly ? y - (G.oy + cy * G.h) : 0.f;
    c.wz = c.clz ? z - (G.oz + cz * G.h) : 0.f;
    return c;
}
template <bool GRAD>
__device__ __forceinline__ float grid_blend(const DGrid& G, float k_wall, const GridCell& c, const float4 lo, const float4 hi,
                                            float& gx, float& gy, float& gz) {
    const float v000 = lo.x, v001 = lo.y, v010 = lo.z, v011 = lo.w, v100 = hi.x, v101 = hi.y, v110 = hi.z, v111 = hi.w;
    const float d00 = v001 - v000, d01 = v011 - v010, d10 = v101 - v100, d11 = v111 - v110;
    const float a00 = fmaf(c.fx, d00, v000), a01 = fmaf(c.fx, d01, v010), a10 = fmaf(c.fx, d10, v100), a11 = fmaf(c.fx, d11, v110);
    const float e0 = a01 - a00, e1 = a11 - a10;
    const float b0 = fmaf(c.fy, e0, a00), b1 = fmaf(c.fy, e1, a10);
    float e = fmaf(c.fz, b1 - b0, b0);
    if (c.clx | c.cly | c.clz) e += k_wall * (c.wx * c.wx + c.wy * c.wy + c.wz * c.wz);
    if (GRAD) {
        const float dx0 = fmaf(c.fy, d01 - d00, d00), dx1 = fmaf(c.fy, d11 - d10, d10);
        gx = (c.clx ? 0.f : fmaf(c.fz, dx1 - dx0, dx0) * G.inv_h) + 2.f * k_wall * c.wx;
        gy = (c.cly ? 0.f : fmaf(c.fz, e1 - e0, e0) * G.inv_h) + 2.f * k_wall * c.wy;
        gz = (c.clz ? 0.f : (b1 - b0) * G.inv_h) + 2.f * k_wall * c.wz;
    }
    return e;
}

// ------------------------------------------------------------------ O2: pair function e(s,t,d) and (de/dd)/d
// L = -[d<dmax] exp(-(d-dvdw-mu)^2/(2 sigma^2)) (sign G1); C = -[d<dc] ln(max(d,floor)/dc), dc = 2.6 for
// donor/acceptor pairs else dvdw (G3, G4); H = -[hb, d<3.4] exp(-(d-2.88)^2/(2*0.3^2)).
// ex2/lg2/rsqrt approximations (about 2 ulp) are far inside the 1e-4 relative tolerance.
template <bool GRAD>
__device__ __forceinline__ float pair_energy(const DParams& P, float d2, float dvdw, bool hb, float& s_over_d) {
    const float rinv = rsqrtf(fmaxf(d2, 1e-12f));
    const float d = d2 * rinv;
    float e = 0.f, de = 0.f;
    if (d < P.long_dmax) {
        const float t = d - dvdw - P.long_mu;
        const float g = __expf(-t * t * P.long_inv_two_sigma2);
        e = -P.w_long * g;
        if (GRAD) de = P.w_long * 2.f * t * P.long_inv_two_sigma2 * g;
    }
    const float dc = hb ? P.hb_dclash : dvdw;
    if (d < dc) {
        e -= P.w_clash * __logf(fmaxf(d, P.d_floor) * __frcp_rn(dc));
        if (GRAD && d > P.d_floor) de -= P.w_clash * rinv;
    }
    if (hb && d < P.hb_dmax) {
        const float t = d - P.hb_mu;
        const float g = __expf(-t * t * P.hb_inv_two_sigma2);
        e -= P.w_hbond * g;
        if (GRAD) de += P.w_hbond * 2.f * t * P.hb_inv_two_sigma2 * g;
    }
    s_over_d = de * rinv;
    return e;
}

// ------------------------------------------------------------------ O2: four pairs at a time (the arithmetic of lane_rec)
// Branch-free in the main part so that the four dependency chains interleave (a thread's pairs are otherwise a serial string of
// shared-memory load -> rsqrt -> ex2 latencies): one lg2 for the product of the four clash ratios, the clash force switched by
// one compare pair.  d* = x_a - x_b; c = dvdw + mu, or -1e15 for a slot without a pair, which then adds exactly zero;
// hbw[u] & lbit != 0: slot u is a donor/acceptor pair (a slot group without any skips that term).  Out: s[u] = (de/dd) / d /
// kappa, so that f_a += s (x_a - x_b).
template <bool GRAD, bool ENERGY>
__device__ __forceinline__ void pair_quad(const PairK& K, const float dx[4], const float dy[4], const float dz[4], const float c[4],
                                         const unsigned hbw[4], unsigned lbit, float& eL, float& eC, float& eH, float s[4]) {
    float d[4], rinv[4], q[4], t[4], dc[4];
    if (ENERGY) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            dc[u] = c[u] - K.mu;                                      // clash distance dvdw (negative: no pair)
            if (hbw[u] != 0u) dc[u] = (hbw[u] & lbit) ? K.hb_dclash : dc[u];
        }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const float d2 = fmaf(dx[u], dx[u], fmaf(dy[u], dy[u], fmaf(dz[u], dz[u], 1e-12f)));
        rinv[u] = rsqrt_approx(d2);
        d[u] = d2 * rinv[u];
        t[u] = d[u] - c[u];
        const float w = t[u] * K.nk2;
        float g = ex2_approx(w * t[u]);
        g = d[u] < K.dmax ? g : 0.f;
        s[u] = 0.f;
        if (ENERGY) {
            eL += g;
            q[u] = fmaxf(dc[u] * fminf(rinv[u], K.inv_floor), 1.f);
        }
        if (GRAD) {
            const float in = (t[u] < K.neg_mu && rinv[u] < K.inv_floor) ? 1.f : 0.f;
            s[u] = rinv[u] * fmaf(in, K.nkc * rinv[u], w * g);
        }
    }
    if (ENERGY) eC += lg2_approx((q[0] * q[1]) * (q[2] * q[3]));
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        if (hbw[u] != 0u) {
            if (hbw[u] & lbit) {
                const float th = d[u] - K.hb_mu;
                float gh = ex2_approx(K.hb_nk2 * th * th);
                gh = d[u] < K.hb_dmax ? gh : 0.f;
                if (ENERGY) eH += gh;
                if (GRAD) {
                    s[u] = fmaf(K.kh * th, gh * rinv[u], s[u]);
                    // the clash range of a donor/acceptor pair ends at hb_dclash, not at dvdw: put the term right
                    const bool plain = t[u] < K.neg_mu, hb = d[u] < K.hb_dclash;
                    if (plain != hb && rinv[u] < K.inv_floor) s[u] = fmaf(hb ? K.nkc : -K.nkc, rinv[u] * rinv[u], s[u]);
                }
            }
        }
    }
}
// ------------------------------------------------------------------ receptor term by direct pair sums (S:8(f) NEXT-3)
// The paper's own evaluation (P:103-125, P:353 item 4): e(s_r, t, |x - r_r|) summed over the receptor atoms within the pair
// function's range -- the cells within R.span of the atom's cell, cells and atoms in a fixed order.  No interpolation, no wall.
template <bool GRAD>
// i0, istep: the caller's share of every cell's atoms (the CTA mapping spreads an atom's partners over its lanes).
__device__ __forceinline__ float rec_direct(const RecDev& R, const DParams& P, int type, float x, float y, float z,
                                            float& gx, float& gy, float& gz, int i0 = 0, int istep = 1) {
    const float rt = __ldg(R.radius + type);
    const unsigned char role_t = __ldg(R.role + type);
    const int cx = (int)floorf((x - R.lo[0]) * R.inv_cell), cy = (int)floorf((y - R.lo[1]) * R.inv_cell), cz = (int)floorf((z - R.lo[2]) * R.inv_cell);
    float e = 0.f;
    for (int kz = max(cz - R.span, 0); kz <= min(cz + R.span, R.nc[2] - 1); ++kz)
        for (int ky = max(cy - R.span, 0); ky <= min(cy + R.span, R.nc[1] - 1); ++ky)
            for (int kx = max(cx - R.span, 0); kx <= min(cx + R.span, R.nc[0] - 1); ++kx) {
                const int c = (kz * R.nc[1] + ky) * R.nc[0] + kx;
                const int r1 = __ldg(R.cell_off + c + 1);
                for (int r = __ldg(R.cell_off + c) + i0; r < r1; r += istep) {
                    const float4 a = __ldg(R.atoms + r);
                    const float dx = x - a.x, dy = y - a.y, dz = z - a.z;
                    const float d2 = dx * dx + dy * dy + dz * dz;
                    if (d2 >= R.cut2) continue;
                    const int s = __float_as_int(a.w);
                    const unsigned char role_s = __ldg(R.role + s);
                    const bool hb = ((role_s & 1) && (role_t & 2)) || ((role_s & 2) && (role_t & 1));
                    float sod;
                    e += pair_energy<GRAD>(P, d2, __ldg(R.radius + s) + rt, hb, sod);
                    if (GRAD) { gx = fmaf(sod, dx, gx); gy = fmaf(sod, dy, gy); gz = fmaf(sod, dz, gz); }
                }
            }
    return e;
}

// ------------------------------------------------------------------ a3..a6: one pose evaluation
// In : t[3], unit q[4] (warp-uniform), theta (lane f holds torsion f-1's angle).
// Out: world coordinates x/y/z[J]; per-lane partial energies e_inter / e_intra (warp_sum them);
//      GRAD: gt[3] = dE/dt, gw[3] = dE/domega (uniform), gth = dE/dtheta on lane f (O9).
// sP : per-warp shared scratch, 6 * J * 32 floats.
// M.n_res > 0: the mixture-density term (mdn.cuh) of every atom is added to its receptor term; mdn_par = the ligand's block.
// MDN: the instance that carries the mixture-density term (its prefetch buffers cost ~90 registers: kept out of the other one)
template <int J, bool GRAD, bool MDN>
__device__ __forceinline__ void eval_pose(const Lig<J>& L, const DGrid& G, const DParams& P,
                                          const MdnDev& M, const float4* __restrict__ mdn_par, const RecDev& RD,
                                          const float t[3], const float q[4], float theta,
                                          float x[J], float y[J], float z[J],
                                          float& e_inter, float& e_intra,
                                          float gt[3], float gw[3], float& gth, float* sP) {
    const int lane = threadIdx.x & 31;

    // ---- a3 forward kinematics (O8): world frame (R, p) of this lane's fragment, F_f = F_parent o L_f,
    // L_f = rotation by theta_f about the reference-frame axis (o, u); F_root = (Rot(q), t).
    float R[9], p[3];
    quat_matrix(q, R);
    p[0] = t[0]; p[1] = t[1]; p[2] = t[2];
    if (L.max_depth > 0) {
        float sn, cs;
        sincosf(theta, &sn, &cs);
        const float oc = 1.f - cs;
        float Lm[9];
        Lm[0] = fmaf(oc * L.ux, L.ux, cs);          Lm[1] = fmaf(oc * L.ux, L.uy, -sn * L.uz);  Lm[2] = fmaf(oc * L.ux, L.uz, sn * L.uy);
        Lm[3] = fmaf(oc * L.uy, L.ux, sn * L.uz);   Lm[4] = fmaf(oc * L.uy, L.uy, cs);          Lm[5] = fmaf(oc * L.uy, L.uz, -sn * L.ux);
        Lm[6] = fmaf(oc * L.uz, L.ux, -sn * L.uy);  Lm[7] = fmaf(oc * L.uz, L.uy, sn * L.ux);   Lm[8] = fmaf(oc * L.uz, L.uz, cs);
        const float c0 = L.ox - (Lm[0] * L.ox + Lm[1] * L.oy + Lm[2] * L.oz);     // L_f(x) = Lm x + c
        const float c1 = L.oy - (Lm[3] * L.ox + Lm[4] * L.oy + Lm[5] * L.oz);
        const float c2 = L.oz - (Lm[6] * L.ox + Lm[7] * L.oy + Lm[8] * L.oz);
        for (int d = 1; d <= L.max_depth; ++d) {                                  // parents are final before children read
            float PR[9], pp[3];
#pragma unroll
            for (int i = 0; i < 9; ++i) PR[i] = __shfl_sync(FULL_MASK, R[i], L.parent);
#pragma unroll
            for (int i = 0; i < 3; ++i) pp[i] = __shfl_sync(FULL_MASK, p[i], L.parent);
            if (L.depth == d) {
#pragma unroll
                for (int r = 0; r < 3; ++r) {
                    R[3 * r + 0] = PR[3 * r] * Lm[0] + PR[3 * r + 1] * Lm[3] + PR[3 * r + 2] * Lm[6];
                    R[3 * r + 1] = PR[3 * r] * Lm[1] + PR[3 * r + 1] * Lm[4] + PR[3 * r + 2] * Lm[7];
                    R[3 * r + 2] = PR[3 * r] * Lm[2] + PR[3 * r + 1] * Lm[5] + PR[3 * r + 2] * Lm[8];
                    p[r] = PR[3 * r] * c0 + PR[3 * r + 1] * c1 + PR[3 * r + 2] * c2 + pp[r];
                }
            }
        }
    }
    // atoms: x_a = R_frag(a) r_a + p_frag(a)
#pragma unroll
    for (int j = 0; j < J; ++j) {
        float A[9], b[3];
#pragma unroll
        for (int i = 0; i < 9; ++i) A[i] = __shfl_sync(FULL_MASK, R[i], L.frg[j]);
#pragma unroll
        for (int i = 0; i < 3; ++i) b[i] = __shfl_sync(FULL_MASK, p[i], L.frg[j]);
        x[j] = A[0] * L.rx[j] + A[1] * L.ry[j] + A[2] * L.rz[j] + b[0];
        y[j] = A[3] * L.rx[j] + A[4] * L.ry[j] + A[5] * L.rz[j] + b[1];
        z[j] = A[6] * L.rx[j] + A[7] * L.ry[j] + A[8] * L.rz[j] + b[2];
    }

    // ---- a4 receptor energy: trilinear gather per atom
    float fx[J], fy[J], fz[J];                     // dE/dx_a
    e_inter = 0.f; e_intra = 0.f;
#pragma unroll
    for (int j = 0; j < J; ++j) {
        fx[j] = fy[j] = fz[j] = 0.f;
        if (L.valid[j]) {
            if (RD.atoms) e_inter += rec_direct<GRAD>(RD, P, L.typ[j], x[j], y[j], z[j], fx[j], fy[j], fz[j]);
            else e_inter += grid_interp_packed<GRAD>(G, P.k_wall, L.typ[j], x[j], y[j], z[j], fx[j], fy[j], fz[j]);
        }
        if (MDN && L.valid[j]) mdn_atom(M, mdn_par, L.n, j * L.S + lane, x[j], y[j], z[j], 0, 1, GRAD, e_inter, fx[j], fy[j], fz[j]);
    }

    // ---- a5 intra-ligand pairs: conflict-free rotation schedule, partner data by shuffle, reaction force shuffled back; four
    // rounds at a time through the branch-free four-pair arithmetic (pair_quad), so that their dependency chains interleave
    {
        const PairK K = make_pairk(P);
        float eL = 0.f, eC = 0.f, eH = 0.f;
        int tile = 0;
#pragma unroll
        for (int j1 = 0; j1 < J; ++j1) {
#pragma unroll
            for (int j2 = j1; j2 < J; ++j2, ++tile) {
                const int rb = L.tile_off[tile], re = L.tile_off[tile + 1];
                for (int r = rb; r < re; r += 4) {
                    float dx[4], dy[4], dz[4], c[4], sv[4];
                    unsigned hbw[4];
                    int kk[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const bool in = r + u < re;                // (a round past the end: empty masks)
                        const uint4 rd = __ldg(reinterpret_cast<const uint4*>(L.rounds + (in ? r + u : rb)));
                        const int k = (int)rd.z;
                        kk[u] = k;
                        int src = lane + k; if (src >= L.S) src -= L.S;
                        const float bx = __shfl_sync(FULL_MASK, x[j2], src);
                        const float by = __shfl_sync(FULL_MASK, y[j2], src);
                        const float bz = __shfl_sync(FULL_MASK, z[j2], src);
                        const float br = __shfl_sync(FULL_MASK, L.rad[j2], src);
                        const bool on = in && ((rd.x >> lane) & 1u);
                        dx[u] = x[j1] - bx; dy[u] = y[j1] - by; dz[u] = z[j1] - bz;
                        c[u] = on ? (L.rad[j1] + br) + K.mu : -1e15f;
                        hbw[u] = (on && ((rd.y >> lane) & 1u)) ? 1u : 0u;
                    }
                    pair_quad<GRAD, true>(K, dx, dy, dz, c, hbw, 1u, eL, eC, eH, sv);
                    if (GRAD) {
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const float s = K.kappa * sv[u];
                            const float px = s * dx[u], py = s * dy[u], pz = s * dz[u];
                            fx[j1] += px; fy[j1] += py; fz[j1] += pz;
                            int dst = lane - kk[u]; if (dst < 0) dst += L.S;
                            fx[j2] -= __shfl_sync(FULL_MASK, px, dst);
                            fy[j2] -= __shfl_sync(FULL_MASK, py, dst);
                            fz[j2] -= __shfl_sync(FULL_MASK, pz, dst);
                        }
                    }
                }
            }
        }
        e_intra += fmaf(K.w_clash_ln2, eC, -fmaf(K.w_long, eL, K.w_hbond * eH));
    }

    if (!GRAD) return;

    // ---- a6 reverse mode through the tree (O9).  Per atom (force, moment about t); inclusive prefix sums over the
    // internal (depth-first) atom order; a torsion's subtree is one contiguous range, so its sums are a difference.
    const int NP = J * 32;
    float carry[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int j = 0; j < J; ++j) {
        float v[6];
        const float ax = x[j] - t[0], ay = y[j] - t[1], az = z[j] - t[2];
        v[0] = L.valid[j] ? fx[j] : 0.f;
        v[1] = L.valid[j] ? fy[j] : 0.f;
        v[2] = L.valid[j] ? fz[j] : 0.f;
        v[3] = L.valid[j] ? ay * fz[j] - az * fy[j] : 0.f;
        v[4] = L.valid[j] ? az * fx[j] - ax * fz[j] : 0.f;
        v[5] = L.valid[j] ? ax * fy[j] - ay * fx[j] : 0.f;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
            for (int c = 0; c < 6; ++c) {
                const float u = __shfl_up_sync(FULL_MASK, v[c], o);
                if (lane >= o) v[c] += u;
            }
        }
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            v[c] += carry[c];
            if (L.valid[j]) sP[c * NP + j * L.S + lane] = v[c];
            carry[c] = __shfl_sync(FULL_MASK, v[c], 31);
        }
    }
    __syncwarp();
    gt[0] = carry[0]; gt[1] = carry[1]; gt[2] = carry[2];
    gw[0] = carry[3]; gw[1] = carry[4]; gw[2] = carry[5];
    gth = 0.f;
    if (lane >= 1 && lane <= L.T) {
        float s[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) s[c] = sP[c * NP + L.hi - 1] - (L.lo > 0 ? sP[c * NP + L.lo - 1] : 0.f);
        // world axis u = R u_ref, axis point b = R o + p (both invariant under this fragment's own torsion)
        const float wx = R[0] * L.ux + R[1] * L.uy + R[2] * L.uz;
        const float wy = R[3] * L.ux + R[4] * L.uy + R[5] * L.uz;
        const float wz = R[6] * L.ux + R[7] * L.uy + R[8] * L.uz;
        const float bx = R[0] * L.ox + R[1] * L.oy + R[2] * L.oz + p[0] - t[0];
        const float by = R[3] * L.ox + R[4] * L.oy + R[5] * L.oz + p[1] - t[1];
        const float bz = R[6] * L.ox + R[7] * L.oy + R[8] * L.oz + p[2] - t[2];
        const float tx = s[3] - (by * s[2] - bz * s[1]);     // torque about b = M_t - (b - t) x F
        const float ty = s[4] - (bz * s[0] - bx * s[2]);
        const float tz = s[5] - (bx * s[1] - by * s[0]);
        gth = wx * tx + wy * ty + wz * tz;
    }
    __syncwarp();
}
