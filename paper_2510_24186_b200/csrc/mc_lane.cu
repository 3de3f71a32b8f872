// mc_lane.cu -- the throughput form of the fused per-chain Monte Carlo kernel (steps a1..a8, a10): one LANE per
// chain, one CTA = up to 128 chains of ONE ligand.
//
// Why a second mapping.  With a warp per chain (mc_kernel.cu) a 30-atom ligand costs ~2,100 warp instructions per
// pose evaluation: partner coordinates and reaction forces travel by shuffles, a third of the lanes idle in every
// pair round, the tree passes are scans, and the scalar work (Philox, Adam, quaternions) is replicated 32 times.
// When there are far more chains than lanes (screens: 0.5-4 M chains), every lane gets its own chain: the ligand
// topology is warp-uniform (staged once per CTA in shared memory and read as broadcasts), every loop bound and
// every topology branch is uniform, and the only divergence left is the distance cut-offs.
//
// Shared memory per CTA: topology {ref xyz + radius, atom meta, fragment records, pair stream} + per chain,
// slot-major ([slot][chain], lanes hit distinct banks): coordinates X[3n], a scratch region W and the current /
// proposed torsion angles.  There is NO per-atom force array.  The reverse pass works on per-fragment wrenches
// (force, moment about the origin): grid forces are summed per fragment as they are produced; a pair force is
// central, so it exerts exactly opposite wrenches on its two atoms -- the stream groups pairs into (atom tile of
// one fragment) x (partner atoms of one other fragment) runs, a run's wrench is accumulated in registers from the
// tile side and applied once as +W to the tile's fragment and -W to the partner's.  The rigid pose, its Adam
// moments and the energies live in registers; the best pose goes to global memory when it improves.
// No atomics anywhere: results are bit-reproducible.
//
// P:N = PAPER.md line N; O*/G* = DESIGN.md section 3.
#include "chain.cuh"
#include "mdn.cuh"

struct LaneTopo {
    const float4* ref;      // [n] {ref x, y, z, vdW radius}
    const int* meta;        // [n] type | (first own atom of its fragment) << 8 | pre-order fragment << 16
    const LaneFrag* frag;   // [T + 1]
    const uint4* stream;    // pair instruction stream: header units (internal.h)
    const float4* rec_c;    // pair records: c[4] per record ...
    const uint32_t* rec_m;  // ... and 3 b | hbmask << 16
    int n, T;
};

// Stage one ligand's topology into shared memory; returns the first byte after it (16-byte aligned).  The pair
// records take their parameter- and launch-dependent form here (internal.h): c = dvdw + mu, and one word
// rec_scale * b | hbmask << 16 -- rec_scale * b is where the coordinates of partner atom b start in the chain's
// coordinate store (3 C floats per atom in shared memory, 3 columns in tensor memory), so the record loop adds it to a
// base and loads.  One pad record (no pairs, atom 0) follows the last one: the loop always fetches one record ahead.
__device__ __forceinline__ unsigned char* lane_stage(LaneTopo& S, unsigned char* smem, const LigHdr* __restrict__ h,
                                                     const float4* __restrict__ atom_f4, const int* __restrict__ atom_i,
                                                     const LaneFrag* __restrict__ lane_frags, const uint4* __restrict__ lane_stream,
                                                     const LaneRec* __restrict__ lane_recs, const DParams& P, int tid, int nt,
                                                     uint32_t rec_scale) {
    const int n = h->n, T = h->T, ls = h->ls_len, nr = h->n_rec;
    float4* ref = reinterpret_cast<float4*>(smem);
    int* meta = reinterpret_cast<int*>(smem + 16 * (size_t)n);
    int* frag = reinterpret_cast<int*>(smem + 16 * (size_t)n + 16 * (size_t)((n + 3) / 4));
    uint4* stream = reinterpret_cast<uint4*>(reinterpret_cast<unsigned char*>(frag) + sizeof(LaneFrag) * (size_t)(T + 1));
    float4* rec_c = reinterpret_cast<float4*>(stream + ls);
    uint32_t* rec_m = reinterpret_cast<uint32_t*>(rec_c + nr + 1);
    const LaneFrag* fsrc = lane_frags + h->frag_off;
    for (int i = tid; i < n; i += nt) ref[i] = __ldg(atom_f4 + h->atom_off + i);
    for (int i = tid; i < (T + 1) * (int)(sizeof(LaneFrag) / 4); i += nt) frag[i] = __ldg(reinterpret_cast<const int*>(fsrc) + i);
    for (int g = tid; g <= T; g += nt) {                     // atom meta from the fragment records
        const int lo = __ldg(&fsrc[g].lo), hi = __ldg(&fsrc[g].own_hi);
        for (int a = lo; a < hi; ++a) meta[a] = (__ldg(atom_i + h->atom_off + a) & 0xff) | ((a == lo) << 8) | (g << 16);
    }
    for (int i = tid; i < ls; i += nt) stream[i] = __ldg(lane_stream + h->ls_off + i);
    for (int i = tid; i <= nr; i += nt) {
        if (i == nr) { rec_c[i] = make_float4(-1e15f, -1e15f, -1e15f, -1e15f); rec_m[i] = 0u; continue; }
        const uint4* src = reinterpret_cast<const uint4*>(lane_recs + h->rec_off + i);
        const uint4 dv = __ldg(src), mt = __ldg(src + 1);
        const float d[4] = {__uint_as_float(dv.x), __uint_as_float(dv.y), __uint_as_float(dv.z), __uint_as_float(dv.w)};
        float c[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) c[k] = d[k] >= 0.f ? d[k] + P.long_mu : -1e15f;
        rec_c[i] = make_float4(c[0], c[1], c[2], c[3]);
        rec_m[i] = rec_scale * mt.x | (mt.y << 16);
    }
    S.ref = ref; S.meta = meta; S.frag = reinterpret_cast<const LaneFrag*>(frag); S.stream = stream; S.rec_c = rec_c; S.rec_m = rec_m; S.n = n; S.T = T;
    return smem + lane_topo_bytes(n, T, ls, nr);
}

// ------------------------------------------------------------------ the coordinates of one chain
// Shared memory, slot-major (slot i of this lane's chain is X[i * C], C = chains per CTA, a compile-time constant so
// that every slot offset is an immediate) -- or TENSOR MEMORY: 256 KB per SM that nothing else on this path uses.  A CTA
// of four warps owns `cols` columns of all 128 TMEM lanes; lane = chain, column 3a + c = coordinate c of atom a, moved
// with tcgen05.st / tcgen05.ld (32x32b: every thread of a warp touches its own lane).  Taking the coordinates (two thirds
// of a chain's shared memory) out of shared memory lets 12 warps stay resident per SM where the shared-memory form holds
// 6-10 (measured: on par overall; an explicit option).
// get(off, ...) takes the atom's offset in the store's own unit, off = kScale * a (what the pair records carry).
// A tensor-memory load is asynchronous: fence() (tcgen05.wait::ld, tied to the destination registers) must sit between
// get() and the first use.
template <int C>
struct XShared {
    static constexpr int kC = C;
    static constexpr uint32_t kScale = 3u * C;
    float* X;
    __device__ __forceinline__ void put(int a, float x, float y, float z) const { float* xa = X + 3 * a * C; xa[0] = x; xa[C] = y; xa[2 * C] = z; }
    __device__ __forceinline__ void get(uint32_t off, float& x, float& y, float& z) const { const float* xa = X + off; x = xa[0]; y = xa[C]; z = xa[2 * C]; }
    __device__ __forceinline__ void fence(float&, float&, float&) const {}
    __device__ __forceinline__ void flush() const {}
};
struct XTensor {
    static constexpr int kC = 32;
    static constexpr uint32_t kScale = 3u;
    uint32_t tb;            // TMEM address of column 0 in this warp's lane quarter
    // writes columns 3a .. 3a+3: atoms are placed in ascending order, so the fourth column is rewritten by atom a + 1
    __device__ __forceinline__ void put(int a, float x, float y, float z) const {
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                     :: "r"(tb + 3u * (uint32_t)a), "r"(__float_as_uint(x)), "r"(__float_as_uint(y)), "r"(__float_as_uint(z)), "r"(0u) : "memory");
    }
    __device__ __forceinline__ void get(uint32_t off, float& x, float& y, float& z) const {
        uint32_t r0, r1, r2, r3;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(tb + off) : "memory");
        x = __uint_as_float(r0); y = __uint_as_float(r1); z = __uint_as_float(r2);
    }
    __device__ __forceinline__ void fence(float& x, float& y, float& z) const {
        asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(x), "+f"(y), "+f"(z) :: "memory");
    }
    __device__ __forceinline__ void flush() const { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
};

// ------------------------------------------------------------------ a3 forward kinematics (O8)
// Fragment frames F_g = F_parent o L_g in pre-order; the frame of a fragment at depth d that has children is kept
// in frame slot d (12 floats of the scratch region), so a child finds its parent at slot depth - 1.  Every fragment
// places its own atoms while its frame is in registers.  th[g - 1] is the torsion angle of fragment g.
template <class XS>
__device__ __forceinline__ void lane_place(const LaneTopo& S, const float R[9], const float p[3], int lo, int hi, const XS& X) {
    for (int a = lo; a < hi; ++a) {
        const float4 r = S.ref[a];
        X.put(a, fmaf(R[0], r.x, fmaf(R[1], r.y, fmaf(R[2], r.z, p[0]))), fmaf(R[3], r.x, fmaf(R[4], r.y, fmaf(R[5], r.z, p[1]))),
              fmaf(R[6], r.x, fmaf(R[7], r.y, fmaf(R[8], r.z, p[2]))));
    }
}
template <class XS>
__device__ __forceinline__ void lane_fk(const LaneTopo& S, const float t[3], const float q[4], const float* __restrict__ th,
                                        const XS& X, float* __restrict__ FR) {
    constexpr int C = XS::kC;
    float R[9], p[3];
    quat_matrix(q, R);
    p[0] = t[0]; p[1] = t[1]; p[2] = t[2];
    if (S.T > 0) {
#pragma unroll
        for (int i = 0; i < 9; ++i) FR[i * C] = R[i];
#pragma unroll
        for (int i = 0; i < 3; ++i) FR[(9 + i) * C] = p[i];
    }
    lane_place(S, R, p, 0, S.frag[0].own_hi, X);
    for (int g = 1; g <= S.T; ++g) {
        const LaneFrag& r = S.frag[g];
        const float ux = r.ux, uy = r.uy, uz = r.uz, ox = r.ox, oy = r.oy, oz = r.oz;
        float sn, cs;
        __sincosf(th[(g - 1) * C], &sn, &cs);
        const float oc = 1.f - cs;
        float Lm[9];
        Lm[0] = fmaf(oc * ux, ux, cs);        Lm[1] = fmaf(oc * ux, uy, -sn * uz);  Lm[2] = fmaf(oc * ux, uz, sn * uy);
        Lm[3] = fmaf(oc * uy, ux, sn * uz);   Lm[4] = fmaf(oc * uy, uy, cs);        Lm[5] = fmaf(oc * uy, uz, -sn * ux);
        Lm[6] = fmaf(oc * uz, ux, -sn * uy);  Lm[7] = fmaf(oc * uz, uy, sn * ux);   Lm[8] = fmaf(oc * uz, uz, cs);
        const float c0 = ox - (Lm[0] * ox + Lm[1] * oy + Lm[2] * oz);         // L_g(x) = Lm x + c
        const float c1 = oy - (Lm[3] * ox + Lm[4] * oy + Lm[5] * oz);
        const float c2 = oz - (Lm[6] * ox + Lm[7] * oy + Lm[8] * oz);
        const int depth = r.depth;
        const float* PF = FR + 12 * (depth - 1) * C;
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
        if (g < S.T && S.frag[g + 1].depth > depth) {      // the next fragment in pre-order is a child: keep the frame
            float* MF = FR + 12 * depth * C;
#pragma unroll
            for (int i = 0; i < 9; ++i) MF[i * C] = R[i];
#pragma unroll
            for (int i = 0; i < 3; ++i) MF[(9 + i) * C] = p[i];
        }
        lane_place(S, R, p, r.lo, r.own_hi, X);
    }
    X.flush();
}

// ------------------------------------------------------------------ a4 receptor energy (O5)
// One 32-byte record of the cell-packed grid per atom (a 256-bit load).  The common case -- the atom lies inside the grid -- takes a short
// path (u = x * inv_h - origin * inv_h by one FMA, floor, fraction, one unsigned range test per axis); an atom on or
// beyond the boundary takes the general clamp of O5 and raises c.cl (bit i: axis i clamped), which sends the blend
// through the wall terms (G8).
// the 32-byte cell record (DGrid::gp) by one 256-bit load
__device__ __forceinline__ void ldg_cell(const float4* p, float4& lo, float4& hi) {
    asm("ld.global.nc.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=f"(lo.x), "=f"(lo.y), "=f"(lo.z), "=f"(lo.w), "=f"(hi.x), "=f"(hi.y), "=f"(hi.z), "=f"(hi.w) : "l"(p));
}
struct LaneCell {
    const float4* p;
    float fx, fy, fz;
    int cl;
};
struct LaneGridK { float nox, noy, noz; };        // -origin * inv_h
__device__ __forceinline__ LaneCell lane_locate(const DGrid& G, const LaneGridK& Q, int type, float x, float y, float z) {
    LaneCell c;
    const float ux = fmaf(x, G.inv_h, Q.nox), uy = fmaf(y, G.inv_h, Q.noy), uz = fmaf(z, G.inv_h, Q.noz);
    int ix = __float2int_rd(ux), iy = __float2int_rd(uy), iz = __float2int_rd(uz);
    c.fx = ux - (float)ix; c.fy = uy - (float)iy; c.fz = uz - (float)iz;
    c.cl = 0;
    if ((unsigned)ix > (unsigned)(G.nx - 2) || (unsigned)iy > (unsigned)(G.ny - 2) || (unsigned)iz > (unsigned)(G.nz - 2)) {
        const float vx = (x - G.ox) * G.inv_h, vy = (y - G.oy) * G.inv_h, vz = (z - G.oz) * G.inv_h;
        const float cx = fminf(fmaxf(vx, 0.f), (float)(G.nx - 1));
        const float cy = fminf(fmaxf(vy, 0.f), (float)(G.ny - 1));
        const float cz = fminf(fmaxf(vz, 0.f), (float)(G.nz - 1));
        ix = min((int)cx, G.nx - 2); iy = min((int)cy, G.ny - 2); iz = min((int)cz, G.nz - 2);
        c.fx = cx - (float)ix; c.fy = cy - (float)iy; c.fz = cz - (float)iz;
        c.cl = (cx != vx ? 1 : 0) | (cy != vy ? 2 : 0) | (cz != vz ? 4 : 0);
    }
    c.p = G.gp + 2 * ((size_t)type * G.plane + ((size_t)iz * G.ny + iy) * G.nx + ix);
    return c;
}
// value, and (grad, warp-uniform) the gradient in GRID units: the caller multiplies by inv_h
__device__ __forceinline__ float lane_blend(const DGrid& G, float k_wall, const LaneCell& c, const float4 lo, const float4 hi, bool grad,
                                            float x, float y, float z, float& gx, float& gy, float& gz) {
    const float v000 = lo.x, v001 = lo.y, v010 = lo.z, v011 = lo.w, v100 = hi.x, v101 = hi.y, v110 = hi.z, v111 = hi.w;
    const float d00 = v001 - v000, d01 = v011 - v010, d10 = v101 - v100, d11 = v111 - v110;
    const float a00 = fmaf(c.fx, d00, v000), a01 = fmaf(c.fx, d01, v010), a10 = fmaf(c.fx, d10, v100), a11 = fmaf(c.fx, d11, v110);
    const float e0 = a01 - a00, e1 = a11 - a10;
    const float b0 = fmaf(c.fy, e0, a00), b1 = fmaf(c.fy, e1, a10);
    float e = fmaf(c.fz, b1 - b0, b0);
    if (grad) {
        const float dx0 = fmaf(c.fy, d01 - d00, d00), dx1 = fmaf(c.fy, d11 - d10, d10);
        gx = fmaf(c.fz, dx1 - dx0, dx0);
        gy = fmaf(c.fz, e1 - e0, e0);
        gz = b1 - b0;
    }
    if (c.cl) {                                   // rare: outside the grid -- clamped axes have no gradient, quadratic wall
        const float vx = (x - G.ox) * G.inv_h, vy = (y - G.oy) * G.inv_h, vz = (z - G.oz) * G.inv_h;
        const float cx = fminf(fmaxf(vx, 0.f), (float)(G.nx - 1));
        const float cy = fminf(fmaxf(vy, 0.f), (float)(G.ny - 1));
        const float cz = fminf(fmaxf(vz, 0.f), (float)(G.nz - 1));
        const float wx = (c.cl & 1) ? x - (G.ox + cx * G.h) : 0.f;
        const float wy = (c.cl & 2) ? y - (G.oy + cy * G.h) : 0.f;
        const float wz = (c.cl & 4) ? z - (G.oz + cz * G.h) : 0.f;
        e += k_wall * (wx * wx + wy * wy + wz * wz);
        if (grad) {
            const float kw = 2.f * k_wall * G.h;
            gx = ((c.cl & 1) ? 0.f : gx) + kw * wx;
            gy = ((c.cl & 2) ? 0.f : gy) + kw * wy;
            gz = ((c.cl & 4) ? 0.f : gz) + kw * wz;
        }
    }
    return e;
}

// All atoms of the ligand, software-pipelined LANE_GD deep: an atom's cell is located and its two records are requested
// LANE_GD - 1 atoms before it is blended, so that the L2 round trip (the wait for it was 11-15 % of the kernel's time
// when an atom was consumed one blend after its request) is covered by the blends of the atoms before it.
// grad (warp-uniform): WR[g] <- wscale * wrench (force, moment about the origin) of the grid forces on the own atoms
// of fragment g, for every g (this initialises WR); wscale = inv_h / kappa (the reverse pass works in the pair terms'
// kappa units, lane_backward).
// The kernel's code must stay small (instruction cache, B300_MICROARCH.md), so there is ONE copy of the evaluation with
// a warp-uniform `grad` flag instead of two template instances.
#ifndef LANE_GD
#define LANE_GD 2     // measured on C5: 2 in flight 225 ms, 3: 238 ms, 4: 245 ms (8,192 ligands) -- the unrolled copies cost more
#endif                // instruction-cache misses than the deeper prefetch saves
// MDN: the mixture-density term of every atom (mdn.cuh) is added where its grid value is blended.
template <bool MDN, class XS>
__device__ __forceinline__ float lane_grid(const LaneTopo& S, const DGrid& G, float k_wall, bool grad, float wscale,
                                           const MdnDev& M, const float4* __restrict__ mdn_par, const XS& X, float* __restrict__ WR) {
    constexpr int C = XS::kC;
    constexpr int GD = MDN ? 1 : LANE_GD;                       // with the term: one copy of mdn_atom, and its registers
    const LaneGridK Q = {-G.ox * G.inv_h, -G.oy * G.inv_h, -G.oz * G.inv_h};
    float e_inter = 0.f;
    float acc[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    int gcur = 0;
    const int n = S.n;
    float x[GD], y[GD], z[GD];
    int m[GD];
    LaneCell c[GD];
    float4 lo[GD], hi[GD];
#pragma unroll
    for (int k = 0; k < GD - 1; ++k) {                    // prologue: atoms 0 .. GD-2 (the tail repeats the last atom)
        const int a = min(k, n - 1);
        m[k] = S.meta[a];
        X.get(XS::kScale * (uint32_t)a, x[k], y[k], z[k]);
        X.fence(x[k], y[k], z[k]);
        c[k] = lane_locate(G, Q, m[k] & 0xff, x[k], y[k], z[k]);
        ldg_cell(c[k].p, lo[k], hi[k]);
    }
    for (int a0 = 0; a0 < n; a0 += GD) {
#pragma unroll
        for (int k = 0; k < GD; ++k) {
            {                                                   // request atom a0 + k + GD - 1 into the slot freed last
                constexpr int D1 = GD - 1;
                const int sl = (k + D1) % GD;
                const int a = min(a0 + k + D1, n - 1);
                m[sl] = S.meta[a];
                X.get(XS::kScale * (uint32_t)a, x[sl], y[sl], z[sl]);
                X.fence(x[sl], y[sl], z[sl]);
                c[sl] = lane_locate(G, Q, m[sl] & 0xff, x[sl], y[sl], z[sl]);
                ldg_cell(c[sl].p, lo[sl], hi[sl]);
            }
            if (a0 + k < n) {                                   // blend atom a0 + k
                float gx, gy, gz;
                e_inter += lane_blend(G, k_wall, c[k], lo[k], hi[k], grad, x[k], y[k], z[k], gx, gy, gz);
                if (MDN) {
                    float me = 0.f, mx = 0.f, my = 0.f, mz = 0.f;
                    mdn_atom(M, mdn_par, n, a0 + k, x[k], y[k], z[k], 0, 1, grad, me, mx, my, mz);
                    e_inter += me;
                    if (grad) { gx = fmaf(mx, G.h, gx); gy = fmaf(my, G.h, gy); gz = fmaf(mz, G.h, gz); }   // grid units, like the blend
                }
                if (grad) {
                    if ((m[k] & 0x100) && a0 + k > 0) {        // first own atom of the next fragment: the previous one is complete
#pragma unroll
                        for (int j = 0; j < 6; ++j) { WR[(6 * gcur + j) * C] = acc[j] * wscale; acc[j] = 0.f; }
                    }
                    gcur = m[k] >> 16;
                    acc[0] += gx; acc[1] += gy; acc[2] += gz;
                    acc[3] += y[k] * gz - z[k] * gy;
                    acc[4] += z[k] * gx - x[k] * gz;
                    acc[5] += x[k] * gy - y[k] * gx;
                }
            }
        }
    }
    if (grad) {
#pragma unroll
        for (int j = 0; j < 6; ++j) WR[(6 * gcur + j) * C] = acc[j] * wscale;
    }
    return e_inter;
}

// ------------------------------------------------------------------ a5 intra-ligand pairs (O2, O6)
// One record: partner atom b against the 4 slots of a tile, branch-free so that the four evaluations interleave.
//   L = -[d<dmax] exp(-(d-dvdw-mu)^2/(2 sigma^2))  (G1):  eL += [d<dmax] 2^(nk2 t^2),  t = d - c,  c = dvdw + mu
//   C = -[d<dc] ln(max(d,floor)/dc)                (G3, G4):  eC += lg2 of the PRODUCT over the 4 slots of
//       max(dc / max(d,floor), 1) (one lg2 per record; the product is at most (dc/floor)^4),  dc = c - mu, or hb_dclash for
//       a donor/acceptor pair.  The force needs no dc: d < dc is t < -mu (t < hb_dclash - c for a donor/acceptor pair).
//   H = -[hb, d<3.4] exp(-(d-2.88)^2/(2*0.3^2)):  eH += ..., only in records that hold such a pair
// GRAD: f_i += s (x_a - x_b) with s = (de/dd) / d / kappa.  A slot without a pair has c = -1e15 and adds 0.
// The 1e-12 inside the squared distance keeps rsqrt finite for coincident atoms (it moves d by < 1e-12 / 2d).
template <bool GRAD, bool ENERGY>
__device__ __forceinline__ void lane_rec(const PairK& K, const float ax[4], const float ay[4], const float az[4],
                                         float bx, float by, float bz, const float4 c4, unsigned hbmask,
                                         float& eL, float& eC, float& eH, float fx[4], float fy[4], float fz[4]) {
    const float c[4] = {c4.x, c4.y, c4.z, c4.w};
    float dc[4];
    if (ENERGY) {
#pragma unroll
        for (int i = 0; i < 4; ++i) dc[i] = c[i] - K.mu;                 // clash distance dvdw (negative: no pair)
        if (hbmask) {                                                // warp-uniform; about one record in three
#pragma unroll
            for (int i = 0; i < 4; ++i) dc[i] = ((hbmask >> i) & 1u) ? K.hb_dclash : dc[i];
        }
    }
    float dx[4], dy[4], dz[4], d[4], rinv[4], s[4], q[4], t[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        dx[i] = ax[i] - bx; dy[i] = ay[i] - by; dz[i] = az[i] - bz;
        const float d2 = fmaf(dx[i], dx[i], fmaf(dy[i], dy[i], fmaf(dz[i], dz[i], 1e-12f)));
        rinv[i] = rsqrt_approx(d2);
        d[i] = d2 * rinv[i];
        t[i] = d[i] - c[i];
        const float u = t[i] * K.nk2;
        float g = ex2_approx(u * t[i]);
        g = d[i] < K.dmax ? g : 0.f;
        if (ENERGY) {
            eL += g;
            q[i] = fmaxf(dc[i] * fminf(rinv[i], K.inv_floor), 1.f);     // dc / max(d, floor); > 1 inside the clash range
        }
        if (GRAD) {
            // s = rinv (u g - [floor < d < dvdw] kc rinv); a donor/acceptor slot is corrected below
            const float in = (t[i] < K.neg_mu && rinv[i] < K.inv_floor) ? 1.f : 0.f;    // one FSET, no select / predicate chain
            s[i] = rinv[i] * fmaf(in, K.nkc * rinv[i], u * g);
        }
    }
    if (ENERGY) eC += lg2_approx((q[0] * q[1]) * (q[2] * q[3]));
    if (hbmask) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            if ((hbmask >> i) & 1u) {
                const float th = d[i] - K.hb_mu;
                float gh = ex2_approx(K.hb_nk2 * th * th);
                gh = d[i] < K.hb_dmax ? gh : 0.f;
                if (ENERGY) eH += gh;
                if (GRAD) {
                    s[i] = fmaf(K.kh * th, gh * rinv[i], s[i]);
                    // the clash range of a donor/acceptor pair ends at hb_dclash, not at dvdw: put the term right
                    const bool plain = t[i] < K.neg_mu, hb = d[i] < K.hb_dclash;
                    if (plain != hb && rinv[i] < K.inv_floor) s[i] = fmaf(hb ? K.nkc : -K.nkc, rinv[i] * rinv[i], s[i]);
                }
            }
        }
    }
    if (GRAD) {
#pragma unroll
        for (int i = 0; i < 4; ++i) { fx[i] = fmaf(s[i], dx[i], fx[i]); fy[i] = fmaf(s[i], dy[i], fy[i]); fz[i] = fmaf(s[i], dz[i], fz[i]); }
    }
}

#ifdef LANE_F32X2
// Experimental: the same record with the FP32 arithmetic of slot pairs (0,1) and (2,3) as packed
// add / mul / fma.rn.f32x2 on 64-bit register pairs kept from the tile load to the force accumulation.
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk2(float a, float b) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void up2(u64 v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
template <bool GRAD, bool ENERGY>
__device__ __forceinline__ void lane_rec2(const PairK& K, const u64 ax[2], const u64 ay[2], const u64 az[2],
                                          float bx, float by, float bz, const float4 c4, unsigned hbmask,
                                          float& eL, float& eC, float& eH, u64 fx[2], u64 fy[2], u64 fz[2]) {
    const u64 bxx = pk2(bx, bx), byy = pk2(by, by), bzz = pk2(bz, bz);
    const u64 eps2 = pk2(1e-12f, 1e-12f), nk22 = pk2(K.nk2, K.nk2), nkc2 = pk2(K.nkc, K.nkc);
    const float cs[4] = {c4.x, c4.y, c4.z, c4.w};
    float q[4];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const u64 c = pk2(cs[2 * h], cs[2 * h + 1]);
        const u64 dx = sub2(ax[h], bxx), dy = sub2(ay[h], byy), dz = sub2(az[h], bzz);
        const u64 d2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, eps2)));
        float d2a, d2b;
        up2(d2, d2a, d2b);
        const float ra = rsqrt_approx(d2a), rb = rsqrt_approx(d2b);
        const u64 rinv = pk2(ra, rb);
        const u64 d = mul2(d2, rinv);
        const u64 t = sub2(d, c);
        const u64 u = mul2(t, nk22);
        const u64 ut = mul2(u, t);
        float uta, utb, da, db, ta, tb;
        up2(ut, uta, utb); up2(d, da, db); up2(t, ta, tb);
        float ga = ex2_approx(uta), gb = ex2_approx(utb);
        ga = da < K.dmax ? ga : 0.f;
        gb = db < K.dmax ? gb : 0.f;
        if (ENERGY) {
            eL += ga + gb;
            float dca = cs[2 * h] - K.mu, dcb = cs[2 * h + 1] - K.mu;
            if (hbmask) {
                dca = ((hbmask >> (2 * h)) & 1u) ? K.hb_dclash : dca;
                dcb = ((hbmask >> (2 * h + 1)) & 1u) ? K.hb_dclash : dcb;
            }
            q[2 * h] = fmaxf(dca * fminf(ra, K.inv_floor), 1.f);
            q[2 * h + 1] = fmaxf(dcb * fminf(rb, K.inv_floor), 1.f);
        }
        if (GRAD) {
            const float ina = (ta < K.neg_mu && ra < K.inv_floor) ? 1.f : 0.f, inb = (tb < K.neg_mu && rb < K.inv_floor) ? 1.f : 0.f;
            u64 s = mul2(rinv, fma2(pk2(ina, inb), mul2(nkc2, rinv), mul2(u, pk2(ga, gb))));
            if (hbmask) {
                float sa, sb;
                up2(s, sa, sb);
                float sv[2] = {sa, sb};
                const float dv[2] = {da, db}, tv[2] = {ta, tb}, rv[2] = {ra, rb};
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    if ((hbmask >> (2 * h + j)) & 1u) {
                        const float th = dv[j] - K.hb_mu;
                        float gh = ex2_approx(K.hb_nk2 * th * th);
                        gh = dv[j] < K.hb_dmax ? gh : 0.f;
                        if (ENERGY) eH += gh;
                        sv[j] = fmaf(K.kh * th, gh * rv[j], sv[j]);
                        const bool plain = tv[j] < K.neg_mu, hb = dv[j] < K.hb_dclash;
                        if (plain != hb && rv[j] < K.inv_floor) sv[j] = fmaf(hb ? K.nkc : -K.nkc, rv[j] * rv[j], sv[j]);
                    }
                }
                s = pk2(sv[0], sv[1]);
            }
            fx[h] = fma2(s, dx, fx[h]); fy[h] = fma2(s, dy, fy[h]); fz[h] = fma2(s, dz, fz[h]);
        } else if (ENERGY && hbmask) {
            const float dv[2] = {da, db};
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                if ((hbmask >> (2 * h + j)) & 1u) {
                    const float th = dv[j] - K.hb_mu;
                    float gh = ex2_approx(K.hb_nk2 * th * th);
                    eH += dv[j] < K.hb_dmax ? gh : 0.f;
                }
            }
        }
    }
    if (ENERGY) eC += lg2_approx((q[0] * q[1]) * (q[2] * q[3]));
}
#endif

// The record stream is read one record ahead, across run, tile and fragment boundaries: `mt` / (bx, by, bz) always hold
// the NEXT record's word and its partner's coordinates (a dependent load), so no run starts with an exposed load.
struct PairCursor {
    const uint4* hp;        // header units
    const float4* rc;       // record c[4]
    const uint32_t* rm;     // record words; rm[0] is the record in `mt`
    uint32_t mt;
    float bx, by, bz;
};

// One tile: w <= 4 consecutive own atoms a0 .. a0+w-1 of fragment g against n_runs runs of partner atoms.
// GRAD: acc += the wrench the tile's atoms receive; WR[fb] -= each run's wrench (kappa units).
template <bool GRAD, bool ENERGY, class XS>
__device__ __forceinline__ void lane_tile(PairCursor& pc, int a0, int w, int n_runs, const PairK& K,
                                          const XS& X, float* __restrict__ WR,
                                          float acc[6], float& eL, float& eC, float& eH) {
    constexpr int C = XS::kC;
    float ax[4], ay[4], az[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) X.get(XS::kScale * (uint32_t)(a0 + (i < w ? i : 0)), ax[i], ay[i], az[i]);
#pragma unroll
    for (int i = 0; i < 4; ++i) X.fence(ax[i], ay[i], az[i]);
    for (int run = 0; run < n_runs; ++run) {
        const uint4 rh = *pc.hp++;
        const int fb = (int)rh.x;
        const uint32_t* const rend = pc.rm + rh.y;
#ifdef LANE_F32X2
        const u64 pax[2] = {pk2(ax[0], ax[1]), pk2(ax[2], ax[3])}, pay[2] = {pk2(ay[0], ay[1]), pk2(ay[2], ay[3])},
                  paz[2] = {pk2(az[0], az[1]), pk2(az[2], az[3])};
        u64 pfx[2] = {0ull, 0ull}, pfy[2] = {0ull, 0ull}, pfz[2] = {0ull, 0ull};
#endif
        float fx[4], fy[4], fz[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) fx[i] = fy[i] = fz[i] = 0.f;
        do {
            const float4 c4 = *pc.rc++;
            const uint32_t mtn = *++pc.rm;
            float nx, ny, nz;
            X.fence(pc.bx, pc.by, pc.bz);
            X.get(mtn & 0xffffu, nx, ny, nz);
#ifdef LANE_F32X2
            lane_rec2<GRAD, ENERGY>(K, pax, pay, paz, pc.bx, pc.by, pc.bz, c4, pc.mt >> 16, eL, eC, eH, pfx, pfy, pfz);
#else
            lane_rec<GRAD, ENERGY>(K, ax, ay, az, pc.bx, pc.by, pc.bz, c4, pc.mt >> 16, eL, eC, eH, fx, fy, fz);
#endif
            pc.mt = mtn; pc.bx = nx; pc.by = ny; pc.bz = nz;
        } while (pc.rm != rend);
#ifdef LANE_F32X2
        if (GRAD) {
            up2(pfx[0], fx[0], fx[1]); up2(pfx[1], fx[2], fx[3]);
            up2(pfy[0], fy[0], fy[1]); up2(pfy[1], fy[2], fy[3]);
            up2(pfz[0], fz[0], fz[1]); up2(pfz[1], fz[2], fz[3]);
        }
#endif
        if (GRAD) {
            float wv[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                wv[0] += fx[i]; wv[1] += fy[i]; wv[2] += fz[i];
                wv[3] += ay[i] * fz[i] - az[i] * fy[i];
                wv[4] += az[i] * fx[i] - ax[i] * fz[i];
                wv[5] += ax[i] * fy[i] - ay[i] * fx[i];
            }
            float* wb = WR + 6 * fb * C;
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                acc[k] += wv[k];
                wb[k * C] -= wv[k];
            }
        }
    }
}

// All pairs of the ligand.  GRAD: WR[g] (initialised by lane_grid, kappa units) += the pair wrenches.
template <bool GRAD, bool ENERGY, class XS>
__device__ __forceinline__ float lane_pairs(const LaneTopo& S, const PairK& K, const XS& X, float* __restrict__ WR) {
    constexpr int C = XS::kC;
    float eL = 0.f, eC = 0.f, eH = 0.f;
    PairCursor pc;
    pc.hp = S.stream; pc.rc = S.rec_c; pc.rm = S.rec_m;
    pc.mt = pc.rm[0];                                               // the first record (the pad record if there is none)
    X.get(pc.mt & 0xffffu, pc.bx, pc.by, pc.bz);
    for (int g = 0; g <= S.T; ++g) {
        const int n_tiles = (int)(*pc.hp++).x;
        if (n_tiles == 0) continue;
        float acc[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        for (int tl = 0; tl < n_tiles; ++tl) {
            const uint4 h = *pc.hp++;
            lane_tile<GRAD, ENERGY, XS>(pc, (int)h.x, (int)h.y, (int)h.z, K, X, WR, acc, eL, eC, eH);
        }
        if (GRAD) {
            float* wg = WR + 6 * g * C;
#pragma unroll
            for (int k = 0; k < 6; ++k) wg[k * C] += acc[k];
        }
    }
    X.fence(pc.bx, pc.by, pc.bz);                                   // the pad record's load is still in flight
    return fmaf(K.w_clash_ln2, eC, -fmaf(K.w_long, eL, K.w_hbond * eH));
}

// ------------------------------------------------------------------ a3..a5: one pose evaluation by one lane
// In : t[3], unit q[4] (registers), th[(g-1)*C] torsion angles (shared), grad (warp-uniform).
// Out: X (world coordinates), e_inter, e_intra (e_intra of a gradient evaluation only if GE); grad: WR[g] = wrench on the
//      own atoms of fragment g in kappa units (1 / K.kappa of the true wrench).
template <bool GE, bool MDN, class XS>
__device__ __forceinline__ void lane_eval(const LaneTopo& S, const DGrid& G, const DParams& P, const PairK& K, bool grad,
                                          const MdnDev& M, const float4* __restrict__ mdn_par,
                                          const float t[3], const float q[4], const float* __restrict__ th,
                                          const XS& X, float* __restrict__ WR, float& e_inter, float& e_intra) {
    lane_fk(S, t, q, th, X, WR);
    e_inter = lane_grid<MDN>(S, G, P.k_wall, grad, G.inv_h * K.inv_kappa, M, mdn_par, X, WR);
    e_intra = grad ? lane_pairs<true, GE, XS>(S, K, X, WR) : lane_pairs<false, true, XS>(S, K, X, WR);
}

// ------------------------------------------------------------------ a6 reverse mode through the tree (O9)
// Fragments in reverse pre-order: when g is visited WR[g] already holds the wrench of its whole subtree; its torsion
// gradient is u_g . (M - x_b x F) with the axis taken from the world coordinates of its two axis atoms, and the
// wrench moves on to the parent.  WR is in kappa units: `sink(g, dE/dtheta)` and g6 = {dE/dt, dE/domega about t} are
// multiplied by kappa on the way out.
template <class XS, class Sink>
__device__ __forceinline__ void lane_backward(const LaneTopo& S, const float t[3], const XS& X,
                                              float* __restrict__ WR, float kappa, float g6[6], Sink sink) {
    constexpr int C = XS::kC;
    for (int g = S.T; g >= 1; --g) {
        const LaneFrag& r = S.frag[g];
        float w[6];
        float* wg = WR + 6 * g * C;
        float* wp = WR + 6 * r.parent * C;
#pragma unroll
        for (int c = 0; c < 6; ++c) { w[c] = wg[c * C]; wp[c * C] += w[c]; }
        float ax, ay, az, ox, oy, oz;
        X.get(XS::kScale * (uint32_t)(r.axis & 0xff), ax, ay, az);
        X.get(XS::kScale * (uint32_t)((r.axis >> 8) & 0xff), ox, oy, oz);
        X.fence(ax, ay, az); X.fence(ox, oy, oz);
        float ux = ox - ax, uy = oy - ay, uz = oz - az;
        const float un = rsqrtf(ux * ux + uy * uy + uz * uz) * kappa;
        const float mx = w[3] - (oy * w[2] - oz * w[1]);
        const float my = w[4] - (oz * w[0] - ox * w[2]);
        const float mz = w[5] - (ox * w[1] - oy * w[0]);
        sink(g, (ux * mx + uy * my + uz * mz) * un);
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) g6[c] = WR[c * C] * kappa;
    const float fx = g6[0], fy = g6[1], fz = g6[2];
    g6[3] -= t[1] * fz - t[2] * fy;
    g6[4] -= t[2] * fx - t[0] * fz;
    g6[5] -= t[0] * fy - t[1] * fx;
}

// ------------------------------------------------------------------ one chain, start to finish, by one lane
// `live` = false for the padding lanes of a partial warp: they run a copy of the last chain (tensor-memory moves are
// warp-collective) and write nothing.
template <bool MDN, class XS>
__device__ __forceinline__ void lane_chain(const McLaunch& a, const LaneTopo& S, int lig, int chain, bool live, int max_depth,
                                           const XS& X, float* __restrict__ WR, float* __restrict__ THC, float* __restrict__ THP,
                                           float* __restrict__ MV) {
    constexpr int C = XS::kC;
    const DParams& P = a.P;
    const PairK K = make_pairk(P);
    const int T = S.T;
    const float4* mdn_par = MDN ? a.mdn.par + a.mdn.lig_off[lig] : nullptr;
    const size_t cidx = (size_t)lig * a.n_chains + chain;
    const uint2 key = make_uint2((uint32_t)a.seed, (uint32_t)(a.seed >> 32));
    const uint32_t gchain = (uint32_t)(a.chain_base + chain);
    float* g_best = a.pose_best + cidx * a.pose_stride;

    float ct[3], cq[4], ecur = 0.f, ebest = 0.f;
    if (a.init_mode == 2) {                                   // resume: the best pose is already in global memory
        const float* src = a.pose_cur + cidx * a.pose_stride;
        ct[0] = src[0]; ct[1] = src[1]; ct[2] = src[2];
        cq[0] = src[3]; cq[1] = src[4]; cq[2] = src[5]; cq[3] = src[6];
        for (int g = 1; g <= T; ++g) THC[(g - 1) * C] = src[7 + S.frag[g].tor];
        ecur = a.e_cur[cidx]; ebest = a.e_best[cidx];
    } else {
        if (a.init_mode == 1) {
            const float* src = a.init_poses + cidx * a.pose_stride;
            ct[0] = src[0]; ct[1] = src[1]; ct[2] = src[2];
            cq[0] = src[3]; cq[1] = src[4]; cq[2] = src[5]; cq[3] = src[6];
            quat_normalise(cq);
            for (int g = 1; g <= T; ++g) THC[(g - 1) * C] = src[7 + S.frag[g].tor];
        } else {                                              // a1 / O11: Philox initialisation
            const uint4 r2 = philox4x32_10(make_uint4(gchain, 0u, (uint32_t)(a.lig_base + lig), 2u), key);
            const float a0 = u01(r2.x), a1 = u01(r2.y), a2 = u01(r2.z);
            const float rr = a.radius * cbrtf(a0), zz = 2.f * a1 - 1.f, sq = sqrtf(fmaxf(1.f - zz * zz, 0.f));
            float sn, cs;
            sincosf(2.f * PI_F * a2, &sn, &cs);
            ct[0] = a.centre[0] + rr * sq * cs; ct[1] = a.centre[1] + rr * sq * sn; ct[2] = a.centre[2] + rr * zz;
            const uint4 r3 = philox4x32_10(make_uint4(gchain, 0u, (uint32_t)(a.lig_base + lig), 3u), key);
            const float b0 = u01(r3.x), b1 = u01(r3.y), b2 = u01(r3.z);
            const float s1 = sqrtf(1.f - b0), s2 = sqrtf(b0);
            float sn1, cs1, sn2, cs2;
            sincosf(2.f * PI_F * b1, &sn1, &cs1);
            sincosf(2.f * PI_F * b2, &sn2, &cs2);
            cq[0] = s2 * cs2; cq[1] = s1 * sn1; cq[2] = s1 * cs1; cq[3] = s2 * sn2;
            quat_normalise(cq);
            for (int g = 1; g <= T; ++g) {                    // torsion k takes element k % 4 of block 4 + k / 4
                const int k = S.frag[g].tor;
                const uint4 r = philox4x32_10(make_uint4(gchain, 0u, (uint32_t)(a.lig_base + lig), 4u + (uint32_t)(k >> 2)), key);
                const uint32_t w = (k & 3) == 0 ? r.x : (k & 3) == 1 ? r.y : (k & 3) == 2 ? r.z : r.w;
                THC[(g - 1) * C] = PI_F * (2.f * u01(w) - 1.f);
            }
        }
    }
    // One loop over "events": event -1 is the evaluation of the initial pose (a1), events 0.. are MC steps.  There is a
    // single call site of the evaluation (instruction-cache footprint), with a warp-uniform grad flag.
    const bool fresh = a.init_mode != 2;
    for (int s = fresh ? -1 : 0; s < a.n_steps; ++s) {
        const uint32_t step = (uint32_t)(a.first_step + s);
        float pt[3] = {ct[0], ct[1], ct[2]}, pq[4] = {cq[0], cq[1], cq[2], cq[3]};
        int entity = 0;
        float um = 0.f;
        if (s >= 0) {
            // O10: the Metropolis block (purpose 1) and the perturbation block (purpose 0) of this step, drawn by ONE copy of
            // the generator (a loop that is not unrolled: the hot code must stay inside the instruction cache)
            uint4 r = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll 1
            for (uint32_t pz = 0; pz < 2; ++pz) {
                const uint4 v = philox4x32_10(make_uint4(gchain, step, (uint32_t)(a.lig_base + lig), 1u - pz), key);
                if (pz == 0) um = u01(v.x);
                else r = v;
            }
            const float u0 = u01(r.x), u1 = u01(r.y), u2 = u01(r.z), u3 = u01(r.w);
            // a2 / O12: perturb one entity of {translation, rotation, torsion k}
            entity = min((int)(u0 * (float)(T + 2)), T + 1);
            for (int g = 1; g <= T; ++g) {
                const float cur = THC[(g - 1) * C];
                THP[(g - 1) * C] = (S.frag[g].tor == entity - 2) ? PI_F * (2.f * u1 - 1.f) : cur;
            }
            if (entity == 0) {
                pt[0] = fminf(fmaxf(pt[0] + P.pert_trans * (2.f * u1 - 1.f), a.box_min[0]), a.box_max[0]);
                pt[1] = fminf(fmaxf(pt[1] + P.pert_trans * (2.f * u2 - 1.f), a.box_min[1]), a.box_max[1]);
                pt[2] = fminf(fmaxf(pt[2] + P.pert_trans * (2.f * u3 - 1.f), a.box_min[2]), a.box_max[2]);
            } else if (entity == 1) {
                quat_rotate_by(pq, P.pert_rot * (2.f * u1 - 1.f), P.pert_rot * (2.f * u2 - 1.f), P.pert_rot * (2.f * u3 - 1.f));
            }
        } else {
            for (int k = 0; k < T; ++k) THP[k * C] = THC[k * C];
        }

        // a3..a7: n_refine Adam steps on the 6+T tangent components (moments reset every MC step, G12), then (a8) the
        // energy of the refined proposal
        float m[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, v[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        float b1p = 1.f, b2p = 1.f, enew = 0.f;
        for (int rf = (s >= 0 ? 0 : P.n_refine); rf <= P.n_refine; ++rf) {
            const bool grad = rf < P.n_refine;
            float ei, ea;
            lane_eval<false, MDN>(S, a.grid, P, K, grad, a.mdn, mdn_par, pt, pq, THP, X, WR, ei, ea);   // the Adam steps need no energy
            enew = ei + ea;
            if (!grad) break;
            b1p *= P.adam_b1; b2p *= P.adam_b2;
            const float c1 = __fdividef(1.f, 1.f - b1p), c2 = __fdividef(1.f, 1.f - b2p);   // 2-ulp division / square root:
            // far inside the tolerance, and the IEEE forms are slow-path subroutines on the chain's critical path
            const bool keep = rf + 1 < P.n_refine;
            float g6[6];
            lane_backward(S, pt, X, WR, K.kappa, g6, [&](int g, float gk) {   // torsion gradients are consumed as produced
                float mk = 0.f, vk = 0.f;
                if (rf > 0) { mk = MV[2 * (g - 1) * C]; vk = MV[(2 * (g - 1) + 1) * C]; }
                mk = P.adam_b1 * mk + (1.f - P.adam_b1) * gk;
                vk = P.adam_b2 * vk + (1.f - P.adam_b2) * gk * gk;
                if (keep) { MV[2 * (g - 1) * C] = mk; MV[(2 * (g - 1) + 1) * C] = vk; }
                float th = THP[(g - 1) * C] - __fdividef(P.lr * (mk * c1), sqrt_approx(vk * c2) + P.adam_eps);
                if (th >= PI_F) th -= 2.f * PI_F;
                if (th < -PI_F) th += 2.f * PI_F;
                THP[(g - 1) * C] = th;
            });
            float dl[6];
#pragma unroll
            for (int i = 0; i < 6; ++i) {
                m[i] = P.adam_b1 * m[i] + (1.f - P.adam_b1) * g6[i];
                v[i] = P.adam_b2 * v[i] + (1.f - P.adam_b2) * g6[i] * g6[i];
                dl[i] = __fdividef(-P.lr * (m[i] * c1), sqrt_approx(v[i] * c2) + P.adam_eps);
            }
            pt[0] = fminf(fmaxf(pt[0] + dl[0], a.box_min[0]), a.box_max[0]);
            pt[1] = fminf(fmaxf(pt[1] + dl[1], a.box_min[1]), a.box_max[1]);
            pt[2] = fminf(fmaxf(pt[2] + dl[2], a.box_min[2]), a.box_max[2]);
            quat_rotate_by(pq, dl[3], dl[4], dl[5]);
        }

        // a8: Metropolis and best tracking; the initial pose is always "accepted"
        bool accept = true;
        if (s >= 0) {
            accept = isfinite(enew) && (um < expf(-P.beta * (enew - ecur)));
            if (a.trace != nullptr && live) {
                tridsk_trace_rec rec;
                rec.e_prop = enew; rec.e_cur = ecur; rec.u = um; rec.flags = (accept ? 1 : 0) | (entity << 8);
                a.trace[cidx * a.trace_stride + a.trace_off + s] = rec;
            }
        }
        if (accept) {
#pragma unroll
            for (int i = 0; i < 3; ++i) ct[i] = pt[i];
#pragma unroll
            for (int i = 0; i < 4; ++i) cq[i] = pq[i];
            for (int k = 0; k < T; ++k) THC[k * C] = THP[k * C];
            ecur = enew;
            if (s < 0 || enew < ebest) {
                ebest = enew;
                if (live) {
                    g_best[0] = pt[0]; g_best[1] = pt[1]; g_best[2] = pt[2];
                    g_best[3] = pq[0]; g_best[4] = pq[1]; g_best[5] = pq[2]; g_best[6] = pq[3];
                    if (s < 0) for (int e = 7; e < a.pose_stride; ++e) g_best[e] = 0.f;
                    for (int g = 1; g <= T; ++g) g_best[7 + S.frag[g].tor] = THP[(g - 1) * C];
                }
            }
        }
    }

    if (!live) return;
    float* dst = a.pose_cur + cidx * a.pose_stride;
    dst[0] = ct[0]; dst[1] = ct[1]; dst[2] = ct[2];
    dst[3] = cq[0]; dst[4] = cq[1]; dst[5] = cq[2]; dst[6] = cq[3];
    for (int e = 7; e < a.pose_stride; ++e) dst[e] = 0.f;
    for (int g = 1; g <= T; ++g) dst[7 + S.frag[g].tor] = THC[(g - 1) * C];
    a.e_cur[cidx] = ecur; a.e_best[cidx] = ebest;
}

// ------------------------------------------------------------------ the fused MC kernel, one lane per chain
// Coordinates in shared memory: one CTA = C = 32, 64, 96 or 128 chains of ONE ligand (any ligand size that fits); C is a
// template parameter so that every slot offset of the chain's shared-memory state is an immediate.
// MINB = resident 128-thread CTAs per SM the register budget must allow (3: 168 registers, 2: 255): the host picks 255 for
// the size buckets whose shared-memory need keeps at most 8 warps per SM resident anyway, 168 (12 warps) for the rest --
// measured: 12 warps at 168 registers beat 16 warps at 128 (C5 1885 -> 1824 ms), 8 warps at 255 do not (1917 ms).
// With the mixture-density term: always 255 (8 warps) -- at 168 the term's prefetch buffers spill (M3 4.9 s against 3.6 s).
template <int MINB, int C, bool MDN>
__global__ void __launch_bounds__(128, MINB) mc_lane_kernel(const McLaunch a) {
    extern __shared__ __align__(16) unsigned char lane_smem[];
    const int tid = threadIdx.x;
    const int cpl = (a.n_chains + C - 1) / C;                 // CTAs per ligand
    const int lig = a.lig_list[blockIdx.x / cpl];
    const int chain = (blockIdx.x % cpl) * C + tid;
    const LigHdr* h = a.hdr + lig;
    LaneTopo S;
    unsigned char* after = lane_stage(S, lane_smem, h, a.atom_f4, a.atom_i, a.lane_frags, a.lane_stream, a.lane_recs, a.P, tid, C,
                                      XShared<C>::kScale);
    const int max_depth = h->max_depth;
    __syncthreads();
    if (chain >= a.n_chains) return;
    const int n = S.n, T = S.T;
    XShared<C> X;
    X.X = reinterpret_cast<float*>(after) + tid;              // slot-major: slot i of this chain is X[i * C]
    float* WR = X.X + 3 * n * C;                              // frames (forward) / wrenches (reverse)
    float* THC = WR + lane_wslots(T, max_depth) * C;          // current accepted torsions, by pre-order fragment g - 1
    float* THP = THC + T * C;                                 // proposal
    float* MV = THP + T * C;                                  // torsion Adam moments {m, v} (n_refine > 1 only)
    lane_chain<MDN>(a, S, lig, chain, true, max_depth, X, WR, THC, THP, MV);
}

// Coordinates in tensor memory: one CTA = 4 warps, every WARP takes its own work item (ligand, block of 32 chains) and
// stages that ligand's topology into its own quarter of the CTA's shared memory; warp w owns TMEM lanes 32w .. 32w+31.
__global__ void __launch_bounds__(128, 3) mc_lane_tm_kernel(const McLaunch a) {
    extern __shared__ __align__(16) unsigned char lane_smem[];
    __shared__ uint32_t tm_base;
    constexpr int C = 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (warp == 0) {                                          // one warp allocates the CTA's columns
        const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&tm_base);
        if (a.tm_cols == 32) asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 32;" :: "r"(dst) : "memory");
        else if (a.tm_cols == 64) asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 64;" :: "r"(dst) : "memory");
        else asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" :: "r"(dst) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    const int wpl = (a.n_chains + 31) / 32;                   // work items per ligand
    const long long item = (long long)blockIdx.x * 4 + warp, n_items = (long long)a.n_list * wpl;
    const bool work = item < n_items;
    const int lig = a.lig_list[work ? item / wpl : 0];
    const int chain0 = (int)(work ? item % wpl : 0) * 32 + lane;
    const bool live = work && chain0 < a.n_chains;
    const int chain = min(chain0, a.n_chains - 1);
    const LigHdr* h = a.hdr + lig;
    LaneTopo S;
    unsigned char* after = lane_stage(S, lane_smem + (size_t)warp * a.lane_region, h, a.atom_f4, a.atom_i, a.lane_frags, a.lane_stream,
                                      a.lane_recs, a.P, lane, 32, XTensor::kScale);
    const int max_depth = h->max_depth;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    if (work) {                                               // warp-uniform
        const int T = S.T;
        XTensor X;
        X.tb = tm_base + ((uint32_t)(warp * 32) << 16);
        float* WR = reinterpret_cast<float*>(after) + lane;
        float* THC = WR + lane_wslots(T, max_depth) * C;
        float* THP = THC + T * C;
        float* MV = THP + T * C;
        lane_chain<false>(a, S, lig, chain, live, max_depth, X, WR, THC, THP, MV);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) {
        if (a.tm_cols == 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 32;" :: "r"(tm_base) : "memory");
        else if (a.tm_cols == 64) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 64;" :: "r"(tm_base) : "memory");
        else asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" :: "r"(tm_base) : "memory");
    }
}

template <bool MDN> __global__ void score_lane_kernel(const ScoreLaunch a);

// Opt-in shared-memory sizes are per device and per function: done once per device (tridsk_create -> mc_lane_prepare).
template <int MINB, int C, bool MDN>
static cudaError_t lane_prepare_one(size_t max_smem_bytes) {
    cudaError_t e = cudaFuncSetAttribute(mc_lane_kernel<MINB, C, MDN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_smem_bytes);
    // residency is bound by shared memory (the chains' coordinates): take the whole 228 KB, the grid gathers live in L2 anyway
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mc_lane_kernel<MINB, C, MDN>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    return e;
}
cudaError_t mc_lane_prepare(size_t max_smem_bytes) {
    cudaError_t e = lane_prepare_one<3, 32, false>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<3, 64, false>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<3, 96, false>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<3, 128, false>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<2, 32, false>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<2, 64, false>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<2, 96, false>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<2, 128, false>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<2, 32, true>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<2, 64, true>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<2, 96, true>(max_smem_bytes);
    if (e == cudaSuccess) e = lane_prepare_one<2, 128, true>(max_smem_bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(score_lane_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_smem_bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(score_lane_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_smem_bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mc_lane_tm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_smem_bytes - 1024);   // it has 16 static bytes
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mc_lane_tm_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    return e;
}

template <int MINB, bool MDN>
static void lane_launch_c(cudaStream_t s, const McLaunch& a, unsigned blocks, int c, size_t smem_bytes) {
    switch (c) {
        case 32: mc_lane_kernel<MINB, 32, MDN><<<blocks, 32, smem_bytes, s>>>(a); break;
        case 64: mc_lane_kernel<MINB, 64, MDN><<<blocks, 64, smem_bytes, s>>>(a); break;
        case 96: mc_lane_kernel<MINB, 96, MDN><<<blocks, 96, smem_bytes, s>>>(a); break;
        default: mc_lane_kernel<MINB, 128, MDN><<<blocks, 128, smem_bytes, s>>>(a); break;
    }
}
cudaError_t launch_mc_lane(cudaStream_t s, const McLaunch& a, int chains_per_cta, size_t smem_bytes, int minb) {
    const int cpl = (a.n_chains + chains_per_cta - 1) / chains_per_cta;
    const long long blocks = (long long)a.n_list * cpl;
    if (blocks <= 0) return cudaSuccess;
    if (blocks > 0x7fffffffLL || chains_per_cta < 32 || chains_per_cta > 128 || (chains_per_cta & 31)) return cudaErrorInvalidValue;
    if (a.mdn.n_res > 0) lane_launch_c<2, true>(s, a, (unsigned)blocks, chains_per_cta, smem_bytes);   // with the term: 255 registers (mdn_atom's one-ahead pipeline holds two parameter blocks)
    else if (minb == 2) lane_launch_c<2, false>(s, a, (unsigned)blocks, chains_per_cta, smem_bytes);
    else lane_launch_c<3, false>(s, a, (unsigned)blocks, chains_per_cta, smem_bytes);
    return cudaGetLastError();
}

cudaError_t launch_mc_lane_tm(cudaStream_t s, const McLaunch& a) {
    const int wpl = (a.n_chains + 31) / 32;
    const long long items = (long long)a.n_list * wpl, blocks = (items + 3) / 4;
    if (blocks <= 0) return cudaSuccess;
    if (blocks > 0x7fffffffLL || (a.tm_cols != 32 && a.tm_cols != 64 && a.tm_cols != 128) || a.lane_region % 16) return cudaErrorInvalidValue;
    mc_lane_tm_kernel<<<(unsigned)blocks, 128, 4 * (size_t)a.lane_region, s>>>(a);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ tridsk_score_grad, lane form: one lane per pose
// One 32-thread CTA takes up to 32 poses of one ligand (the host groups poses by ligand: seg_*, perm).
template <bool MDN>
__global__ void __launch_bounds__(32) score_lane_kernel(const ScoreLaunch a) {
    extern __shared__ __align__(16) unsigned char lane_smem[];
    constexpr int C = 32;
    const int tid = threadIdx.x;
    const int lig = a.seg_lig[blockIdx.x];
    const LigHdr* h = a.hdr + lig;
    LaneTopo S;
    unsigned char* after = lane_stage(S, lane_smem, h, a.atom_f4, a.atom_i, a.lane_frags, a.lane_stream, a.lane_recs, a.P, tid, 32,
                                      XShared<32>::kScale);
    __syncthreads();
    if (tid >= a.seg_cnt[blockIdx.x]) return;
    const int i = a.perm[a.seg_start[blockIdx.x] + tid];
    const int n = S.n, T = S.T;
    const PairK K = make_pairk(a.P);
    XShared<32> X;
    X.X = reinterpret_cast<float*>(after) + tid;
    float* WR = X.X + 3 * n * C;
    float* TH = WR + lane_wslots(T, h->max_depth) * C;
    const float* src = a.poses + (size_t)i * a.pose_stride;
    float t[3] = {src[0], src[1], src[2]}, q[4] = {src[3], src[4], src[5], src[6]};
    quat_normalise(q);
    for (int g = 1; g <= T; ++g) TH[(g - 1) * C] = src[7 + S.frag[g].tor];
    float ei, ea;
    lane_eval<true, MDN>(S, a.grid, a.P, K, a.grad != nullptr, a.mdn, MDN ? a.mdn.par + a.mdn.lig_off[lig] : nullptr, t, q, TH, X, WR, ei, ea);
    a.energy[3 * (size_t)i] = ei + ea; a.energy[3 * (size_t)i + 1] = ei; a.energy[3 * (size_t)i + 2] = ea;
    if (a.grad != nullptr) {
        float* gr = a.grad + (size_t)i * a.grad_stride;
        for (int e = 6; e < a.grad_stride; ++e) gr[e] = 0.f;
        float g6[6];
        lane_backward(S, t, X, WR, K.kappa, g6, [&](int g, float gk) { gr[6 + S.frag[g].tor] = gk; });
#pragma unroll
        for (int c = 0; c < 6; ++c) gr[c] = g6[c];
    }
    if (a.coords != nullptr) {
        float* c = a.coords + (size_t)i * a.coord_stride * 3;
        for (int p = 0; p < n; ++p) {
            const int orig = (__ldg(a.atom_i + h->atom_off + p) >> 16) & 0xff;
            c[3 * orig] = X.X[3 * p * C]; c[3 * orig + 1] = X.X[(3 * p + 1) * C]; c[3 * orig + 2] = X.X[(3 * p + 2) * C];
        }
        for (int e = 3 * n; e < 3 * a.coord_stride; ++e) c[e] = 0.f;
    }
}

cudaError_t launch_score_lane(cudaStream_t s, const ScoreLaunch& a, int n_seg, size_t smem_bytes) {
    if (n_seg <= 0) return cudaSuccess;
    if (a.mdn.n_res > 0) score_lane_kernel<true><<<n_seg, 32, smem_bytes, s>>>(a);
    else score_lane_kernel<false><<<n_seg, 32, smem_bytes, s>>>(a);
    return cudaGetLastError();
}
