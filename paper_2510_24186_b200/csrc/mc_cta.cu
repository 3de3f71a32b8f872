// mc_cta.cu -- the latency form of the fused per-chain Monte Carlo kernel (steps a1..a8, a10): one CTA per chain.
//
// A single dock has a few hundred chains, each a serial string of thousands of pose evaluations: the time of a dock is
// (evaluations per chain) x (latency of one evaluation), and a warp per chain (mc_kernel.cu) leaves that latency at
// ~2,100 dependent warp instructions.  Here a chain gets 4 warps:
//   * every WARP keeps the whole pose and all fragment frames in registers (lane g = fragment g in pre-order) and
//     repeats the scalar work -- Philox, forward kinematics of the frames, the reverse pass, Adam, Metropolis -- so the
//     warps never have to exchange pose state and take identical decisions by construction;
//   * the atoms are spread over the CTA, `lpa` (8, 4, 2 or 1) lanes per atom: the gradient evaluation walks the pair set in ROW form
//     (every atom meets all its partners, each pair is visited from both ends), so an atom's force is accumulated by
//     its own lanes -- no scatter, no atomics, bit-reproducible; the energy-only evaluation walks the flat pair list;
//   * the receptor term of an atom is two 16-byte gathers whose L2 latency hides behind the pair loop;
//   * two __syncthreads per evaluation: coordinates visible, per-atom (force, moment) / energy partials visible.
// Ligands above 64 atoms: two warps per chain and a dense partner sweep instead of pair records (cta_eval_dense, internal.h),
// so that eight such chains stay resident per SM.
//
// P:N = PAPER.md line N; O*/G* = DESIGN.md section 3.
#include "chain.cuh"
#include "mdn.cuh"

struct CtaTopo {
    const float4* ref;      // [n] {ref x, y, z, vdW radius}, internal (depth-first) atom order
    const int* meta;        // [n] type | pre-order fragment << 8 | original index << 16
    const LaneFrag* frag;   // [T + 1] pre-order
    const int* rows;        // [n + 1] row offsets into recs
    const uint2* recs;      // [2P] row records {b | hb << 8, c}, then [P] flat records {a | b << 8 | hb << 16, c}; c = dvdw + mu
    const uint2* flat;      // the flat records
    const float* tt;        // n > 64: [32][33] c = dvdw + mu of a pair of atom types
    const unsigned* msk;    // n > 64: [4][npad / 32][npad] lanes l of the chunk that are paired with b / form a donor-acceptor pair with b;
                            //         [2], [3]: the same restricted to l < b
    float4* part;           // n > 64: per-warp partial forces [warps][npad]
    float4* X4;             // n > 64: {x, y, z, atom type as int bits} [npad], entries beyond n stay zero
    float *X, *AF, *PF, *red;  // X[3][n], AF[n][8] = {force, 0, moment about t, 0}, PF = its prefix sums, red[64]
    int n, T, P, lpa, npad;
    bool rounds;            // n > 64: dense partner sweep instead of pair records (internal.h)
};

// this lane's fragment (lane g = fragment g in pre-order; lanes beyond T are idle copies of the root)
struct CtaFrag {
    float ux, uy, uz, ox, oy, oz;
    int parent, depth, lo, own_hi, tor, sub_hi;              // sub_hi: end of the subtree's atom range [lo, sub_hi)
    bool valid;
};

__device__ __forceinline__ void cta_stage(CtaTopo& S, CtaFrag& F, unsigned char* smem, const LigHdr* __restrict__ h,
                                          const float4* __restrict__ atom_f4, const int* __restrict__ atom_i,
                                          const LaneFrag* __restrict__ lane_frags, const int* __restrict__ cta_rows,
                                          const uint2* __restrict__ cta_recs, const float* __restrict__ cta_rtab, const DParams& P,
                                          int dense_n) {
    const int n = h->n, T = h->T, np = h->n_pairs, tid = threadIdx.x, nt = blockDim.x, lane = tid & 31;
    const bool rounds = n > dense_n;                             // dense partner sweep (internal.h)
    const CtaLayout L = cta_layout(n, T, np, rounds);
    float4* ref = reinterpret_cast<float4*>(smem + L.ref);
    int* meta = reinterpret_cast<int*>(smem + L.meta);
    int* frag = reinterpret_cast<int*>(smem + L.frag);
    int* rows = reinterpret_cast<int*>(smem + L.rows);
    uint2* recs = reinterpret_cast<uint2*>(smem + L.recs);
    const LaneFrag* fsrc = lane_frags + h->frag_off;
    for (int i = tid; i < n; i += nt) ref[i] = __ldg(atom_f4 + h->atom_off + i);
    for (int i = tid; i < (T + 1) * (int)(sizeof(LaneFrag) / 4); i += nt) frag[i] = __ldg(reinterpret_cast<const int*>(fsrc) + i);
    for (int g = tid; g <= T; g += nt) {
        const int lo = __ldg(&fsrc[g].lo), hi = __ldg(&fsrc[g].own_hi);
        for (int a = lo; a < hi; ++a) {
            const int w = __ldg(atom_i + h->atom_off + a);
            meta[a] = (w & 0xff) | (g << 8) | (((w >> 16) & 0xff) << 16);
        }
    }
    for (int i = tid; i <= n; i += nt) rows[i] = __ldg(cta_rows + h->cta_row_off + i);
    S.tt = nullptr; S.msk = nullptr; S.part = nullptr; S.X4 = nullptr; S.npad = 0;
    if (!rounds) {
        for (int i = tid; i < 3 * np; i += nt) {
            const uint2 r = __ldg(cta_recs + h->cta_rec_off + i);
            recs[i] = make_uint2(r.x, __float_as_uint(__uint_as_float(r.y) + P.long_mu));
        }
    } else {                                                  // no records: the type-pair table, and the masks from the round table
        const int npad = (n + 31) / 32 * 32, nch = npad / 32;
        float* tt = reinterpret_cast<float*>(smem + L.tt);
        float* rad = reinterpret_cast<float*>(smem + L.red);  // scratch until the first evaluation: vdW radius by atom type
        unsigned* mk = reinterpret_cast<unsigned*>(smem + L.masks);
        float4* x4 = reinterpret_cast<float4*>(smem + L.X);
        for (int i = tid; i < 4 * npad * nch; i += nt) mk[i] = 0u;
        for (int i = tid; i < npad; i += nt) x4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int i = tid; i < 32; i += nt) rad[i] = 0.f;
        __syncthreads();                                      // ref, meta staged; scratch zeroed
        for (int i = tid; i < n; i += nt) rad[meta[i] & 31] = ref[i].w;
        __syncthreads();
        for (int i = tid; i < 32 * 32; i += nt) tt[(i >> 5) * 33 + (i & 31)] = (rad[i >> 5] + rad[i & 31]) + P.long_mu;
        const int plane = nch * npad;
        for (int i = tid; i < (n / 2) * n; i += nt) {
            const float d = __ldg(cta_rtab + h->cta_rt_off + i);
            if (d < 0.f) continue;
            const int k = i / n + 1, l = i - (k - 1) * n, b = (l + k) % n;
            const int lo = min(l, b), hi = max(l, b);         // the energy-only sweep meets the pair as (lane lo, partner hi)
            const bool hbp = (__float_as_uint(d) & 1u) != 0u;
            atomicOr(&mk[(l >> 5) * npad + b], 1u << (l & 31));
            atomicOr(&mk[(b >> 5) * npad + l], 1u << (b & 31));
            atomicOr(&mk[2 * plane + (lo >> 5) * npad + hi], 1u << (lo & 31));
            if (hbp) {
                atomicOr(&mk[plane + (l >> 5) * npad + b], 1u << (l & 31));
                atomicOr(&mk[plane + (b >> 5) * npad + l], 1u << (b & 31));
                atomicOr(&mk[3 * plane + (lo >> 5) * npad + hi], 1u << (lo & 31));
            }
        }
        S.tt = tt; S.msk = mk;
        S.part = reinterpret_cast<float4*>(smem + L.part);
        S.X4 = x4;
        S.npad = npad;
    }
    S.rounds = rounds;
    S.flat = recs + 2 * np;
    S.ref = ref; S.meta = meta; S.frag = reinterpret_cast<const LaneFrag*>(frag); S.rows = rows; S.recs = recs;
    S.X = reinterpret_cast<float*>(smem + L.X); S.AF = reinterpret_cast<float*>(smem + L.AF);
    S.PF = reinterpret_cast<float*>(smem + L.PF);
    S.red = reinterpret_cast<float*>(smem + L.red);
    S.n = n; S.T = T; S.P = np;
    int threads;
    cta_shape(n, &threads, &S.lpa);
    __syncthreads();
    const LaneFrag& r = S.frag[lane <= T ? lane : 0];
    F.valid = lane <= T;
    F.ux = r.ux; F.uy = r.uy; F.uz = r.uz; F.ox = r.ox; F.oy = r.oy; F.oz = r.oz;
    F.parent = F.valid ? r.parent : 0; F.depth = F.valid ? r.depth : 0;
    F.lo = r.lo; F.own_hi = F.valid ? r.own_hi : r.lo; F.tor = F.valid ? r.tor : -1;
    int e = lane + 1;
    while (F.valid && e <= T && S.frag[e].depth > r.depth) ++e;      // the subtree of g is the fragment range [g, g_end)
    F.sub_hi = F.valid ? S.frag[e - 1].own_hi : 1;
}

// record form: per-slot flags; a lane without a pair in slot u passes ok[u] = false
template <bool GRAD, bool ENERGY>
__device__ __forceinline__ void cta_pairs4(const PairK& K, const float dx[4], const float dy[4], const float dz[4], const float c_in[4],
                                           const bool hb_in[4], const bool ok[4], float& eL, float& eC, float& eH,
                                           float& fx, float& fy, float& fz) {
    float c[4], s[4];
    unsigned hbw[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { c[u] = ok[u] ? c_in[u] : -1e15f; hbw[u] = (ok[u] && hb_in[u]) ? 1u : 0u; }
    pair_quad<GRAD, ENERGY>(K, dx, dy, dz, c, hbw, 1u, eL, eC, eH, s);
    if (GRAD) {
#pragma unroll
        for (int u = 0; u < 4; ++u) { fx = fmaf(s[u], dx[u], fx); fy = fmaf(s[u], dy[u], fy); fz = fmaf(s[u], dz[u], fz); }
    }
}
// dense partner sweep (internal.h): this lane's atom `me` against four partners; hw.{x,y,z,w} = the lanes that form a
// donor/acceptor pair with partner 0..3 -- a partner without any skips that term for the whole warp
template <bool GRAD, bool ENERGY>
__device__ __forceinline__ void cta_dense4(const PairK& K, const float4 me, const float4 pb[4], const float c[4], const uint4 hw,
                                           unsigned lbit, float& eL, float& eC, float& eH, float& ax, float& ay, float& az) {
    const unsigned hbw[4] = {hw.x, hw.y, hw.z, hw.w};
    float dx[4], dy[4], dz[4], s[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { dx[u] = me.x - pb[u].x; dy[u] = me.y - pb[u].y; dz[u] = me.z - pb[u].z; }
    pair_quad<GRAD, ENERGY>(K, dx, dy, dz, c, hbw, lbit, eL, eC, eH, s);
    if (GRAD) {
#pragma unroll
        for (int u = 0; u < 4; ++u) { ax = fmaf(s[u], dx[u], ax); ay = fmaf(s[u], dy[u], ay); az = fmaf(s[u], dz[u], az); }
    }
}

// ------------------------------------------------------------------ receptor term by direct pair sums, CTA form (S:8(f) NEXT-3)
// e(s_r, t, |x - r_r|) summed over the receptor atoms within the pair function's range (P:103-125, P:353 item 4), for this
// thread's share (i0, i0 + istep, ... of every slice) of the partners of the ligand atom at (x, y, z).  The receptor's cells
// (RecDev) are sorted x fastest, so per (y, z) row of cells within range the candidates are ONE contiguous slice, trimmed to
// the x interval that can still lie inside the cut-off.  The warp walks the rows in lockstep, every lane its own slice of the
// row, one atom per iteration; an atom inside the cut-off goes to a four-slot queue, and when any lane's queue is full all lanes
// evaluate theirs with the branch-free four-pair arithmetic (cta_quad) -- the costly part runs with most lanes busy although
// only one scanned atom in four to ten is in range.  ALL 32 lanes of a warp must call (work = false: nothing to do).
// e += this share of the energy; (fx, fy, fz) += its force in kappa units, like the intra-ligand pair force.
template <bool GRAD, bool ENERGY>
__device__ __forceinline__ void cta_rec_direct(const RecDev& R, const PairK& K, bool work, int type, float x, float y, float z,
                                               int i0, int istep, float& e, float& fx, float& fy, float& fz) {
    const float rt = work ? __ldg(R.radius + type) : 0.f;
    const unsigned role_t = work ? __ldg(R.role + type) : 0u;
    float4 q0 = make_float4(0.f, 0.f, 0.f, 0.f), q1 = q0, q2 = q0, q3 = q0;
    int cnt = 0;
    float eL = 0.f, eC = 0.f, eH = 0.f;
    auto flush = [&]() {
        const float4 qa[4] = {q0, q1, q2, q3};
        float dx[4], dy[4], dz[4], c[4], sv[4];
        unsigned hbw[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const bool valid = u < cnt;
            const int st = valid ? __float_as_int(qa[u].w) : 0;
            const unsigned role_s = __ldg(R.role + st);
            dx[u] = x - qa[u].x; dy[u] = y - qa[u].y; dz[u] = z - qa[u].z;
            c[u] = valid ? (__ldg(R.radius + st) + rt) + K.mu : -1e15f;
            hbw[u] = (valid && (((role_s & 1u) && (role_t & 2u)) || ((role_s & 2u) && (role_t & 1u)))) ? 1u : 0u;
        }
        pair_quad<GRAD, ENERGY>(K, dx, dy, dz, c, hbw, 1u, eL, eC, eH, sv);
        if (GRAD) {
#pragma unroll
            for (int u = 0; u < 4; ++u) { fx = fmaf(sv[u], dx[u], fx); fy = fmaf(sv[u], dy[u], fy); fz = fmaf(sv[u], dz[u], fz); }
        }
        cnt = 0;
    };
    // the rows are walked in lockstep (row offsets -span .. span about every lane's own cell: uniform control flow), the slice of a
    // row differs per lane
    const int cy = __float2int_rd((y - R.lo[1]) * R.inv_cell), cz = __float2int_rd((z - R.lo[2]) * R.inv_cell);
    for (int oz = -R.span; oz <= R.span; ++oz)
        for (int oy = -R.span; oy <= R.span; ++oy) {
            const int ky = cy + oy, kz = cz + oz;
            int r = 0, r1 = 0;
            if (work && (unsigned)ky < (unsigned)R.nc[1] && (unsigned)kz < (unsigned)R.nc[2]) {
                const float y0 = R.lo[1] + R.cell * (float)ky, z0 = R.lo[2] + R.cell * (float)kz;
                const float dy = fmaxf(0.f, fmaxf(y0 - y, y - (y0 + R.cell))), dz = fmaxf(0.f, fmaxf(z0 - z, z - (z0 + R.cell)));
                const float rem = R.cut2 - dy * dy - dz * dz;
                if (rem > 0.f) {
                    const float hx = sqrt_approx(rem) + 1e-3f;       // (a hair wider: the cut-off test below is the exact one)
                    const int kx0 = max(0, __float2int_rd((x - hx - R.lo[0]) * R.inv_cell));
                    const int kx1 = min(R.nc[0] - 1, __float2int_rd((x + hx - R.lo[0]) * R.inv_cell));
                    if (kx0 <= kx1) {
                        const int base = (kz * R.nc[1] + ky) * R.nc[0];
                        r = __ldg(R.cell_off + base + kx0) + i0;
                        r1 = __ldg(R.cell_off + base + kx1 + 1);
                    }
                }
            }
            while (__any_sync(FULL_MASK, r < r1)) {
                if (r < r1) {
                    const float4 a = __ldg(R.atoms + r);
                    r += istep;
                    const float dx = x - a.x, dy = y - a.y, dz = z - a.z;
                    if (dx * dx + dy * dy + dz * dz < R.cut2) {
                        if (cnt == 0) q0 = a; else if (cnt == 1) q1 = a; else if (cnt == 2) q2 = a; else q3 = a;
                        ++cnt;
                    }
                }
                if (__any_sync(FULL_MASK, cnt == 4)) flush();
            }
        }
    if (__any_sync(FULL_MASK, cnt > 0)) flush();
    if (ENERGY) e += fmaf(K.w_clash_ln2, eC, -fmaf(K.w_long, eL, K.w_hbond * eH));
}

// ------------------------------------------------------------------ a3 forward kinematics of the frames (O8)
// World frame (R, p) of this lane's fragment, F_g = F_parent o L_g, by pointer jumping (every warp the same).
__device__ __forceinline__ void cta_frames(const CtaFrag& F, int max_depth, const float t[3], const float q[4], float theta,
                                           float R[9], float p[3]) {
    const int lane = threadIdx.x & 31;
    // ---- a3 forward kinematics (O8): world frame (R, p) of this lane's fragment, F_g = F_parent o L_g, by pointer jumping:
    // every lane starts from its own local transform L_g (the root from the rigid transform) and folds in the accumulated
    // transform of its current ancestor, whose own ancestor it then adopts -- ceil(log2(depth + 1)) rounds instead of `depth`.
    quat_matrix(q, R);
    p[0] = t[0]; p[1] = t[1]; p[2] = t[2];
    if (max_depth > 0) {
        int anc = -1;
        if (F.valid && lane >= 1) {
            float sn, cs;
            __sincosf(theta, &sn, &cs);
            const float oc = 1.f - cs;
            R[0] = fmaf(oc * F.ux, F.ux, cs);          R[1] = fmaf(oc * F.ux, F.uy, -sn * F.uz);  R[2] = fmaf(oc * F.ux, F.uz, sn * F.uy);
            R[3] = fmaf(oc * F.uy, F.ux, sn * F.uz);   R[4] = fmaf(oc * F.uy, F.uy, cs);          R[5] = fmaf(oc * F.uy, F.uz, -sn * F.ux);
            R[6] = fmaf(oc * F.uz, F.ux, -sn * F.uy);  R[7] = fmaf(oc * F.uz, F.uy, sn * F.ux);   R[8] = fmaf(oc * F.uz, F.uz, cs);
            p[0] = F.ox - (R[0] * F.ox + R[1] * F.oy + R[2] * F.oz);
            p[1] = F.oy - (R[3] * F.ox + R[4] * F.oy + R[5] * F.oz);
            p[2] = F.oz - (R[6] * F.ox + R[7] * F.oy + R[8] * F.oz);
            anc = F.parent;
        }
        for (int span = 1; span <= max_depth; span <<= 1) {          // after the round, `2 * span` transforms are folded
            const int src = anc < 0 ? lane : anc;
            float PR[9], pp[3];
#pragma unroll
            for (int i = 0; i < 9; ++i) PR[i] = __shfl_sync(FULL_MASK, R[i], src);
#pragma unroll
            for (int i = 0; i < 3; ++i) pp[i] = __shfl_sync(FULL_MASK, p[i], src);
            const int na = __shfl_sync(FULL_MASK, anc, src);
            if (anc >= 0) {
                float N[9], np3[3];
#pragma unroll
                for (int r = 0; r < 3; ++r) {
                    N[3 * r + 0] = PR[3 * r] * R[0] + PR[3 * r + 1] * R[3] + PR[3 * r + 2] * R[6];
                    N[3 * r + 1] = PR[3 * r] * R[1] + PR[3 * r + 1] * R[4] + PR[3 * r + 2] * R[7];
                    N[3 * r + 2] = PR[3 * r] * R[2] + PR[3 * r + 1] * R[5] + PR[3 * r + 2] * R[8];
                    np3[r] = PR[3 * r] * p[0] + PR[3 * r + 1] * p[1] + PR[3 * r + 2] * p[2] + pp[r];
                }
#pragma unroll
                for (int i = 0; i < 9; ++i) R[i] = N[i];
#pragma unroll
                for (int i = 0; i < 3; ++i) p[i] = np3[i];
                anc = na;
            }
        }
    }
}

// ------------------------------------------------------------------ a6 reverse mode through the tree (O9)
// In: the per-atom (force, moment about t) records AF of the whole ligand (visible).  Out: g6, gth as cta_eval.
__device__ __forceinline__ void cta_reverse(const CtaTopo& S, const CtaFrag& F, const float R[9], const float p[3], const float t[3],
                                            float g6[6], float& gth) {
    const int lane = threadIdx.x & 31, n = S.n;
    // ---- a6 reverse mode through the tree (O9): inclusive prefix sums of the per-atom (force, moment) records over the
    // depth-first atom order (32 atoms per round, shuffle scan + carry); a fragment's subtree is the contiguous atom range
    // [lo, sub_hi), so its wrench is a difference of two prefix entries.  Every warp writes the same prefix values to PF.
    float carry[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    float4* PF = reinterpret_cast<float4*>(S.PF);
    for (int a0 = 0; a0 < n; a0 += 32) {
        const int a = a0 + lane;
        float v[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (a < n) {
            const float4 f = reinterpret_cast<const float4*>(S.AF)[2 * a], mo = reinterpret_cast<const float4*>(S.AF)[2 * a + 1];
            v[0] = f.x; v[1] = f.y; v[2] = f.z; v[3] = mo.x; v[4] = mo.y; v[5] = mo.z;
        }
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
            for (int c = 0; c < 6; ++c) {
                const float u = __shfl_up_sync(FULL_MASK, v[c], o);
                if (lane >= o) v[c] += u;
            }
        }
#pragma unroll
        for (int c = 0; c < 6; ++c) v[c] += carry[c];
        if (a < n) { PF[2 * a] = make_float4(v[0], v[1], v[2], 0.f); PF[2 * a + 1] = make_float4(v[3], v[4], v[5], 0.f); }
#pragma unroll
        for (int c = 0; c < 6; ++c) carry[c] = __shfl_sync(FULL_MASK, v[c], 31);
    }
    __syncwarp();
    float s[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (F.valid) {
        const float4 hf = PF[2 * (F.sub_hi - 1)], hm = PF[2 * (F.sub_hi - 1) + 1];
        s[0] = hf.x; s[1] = hf.y; s[2] = hf.z; s[3] = hm.x; s[4] = hm.y; s[5] = hm.z;
        if (F.lo > 0) {
            const float4 lf = PF[2 * (F.lo - 1)], lm = PF[2 * (F.lo - 1) + 1];
            s[0] -= lf.x; s[1] -= lf.y; s[2] -= lf.z; s[3] -= lm.x; s[4] -= lm.y; s[5] -= lm.z;
        }
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) g6[c] = carry[c];
    gth = 0.f;
    if (F.valid && lane >= 1) {
        const float wx = R[0] * F.ux + R[1] * F.uy + R[2] * F.uz;
        const float wy = R[3] * F.ux + R[4] * F.uy + R[5] * F.uz;
        const float wz = R[6] * F.ux + R[7] * F.uy + R[8] * F.uz;
        const float bx = R[0] * F.ox + R[1] * F.oy + R[2] * F.oz + p[0] - t[0];
        const float by = R[3] * F.ox + R[4] * F.oy + R[5] * F.oz + p[1] - t[1];
        const float bz = R[6] * F.ox + R[7] * F.oy + R[8] * F.oz + p[2] - t[2];
        const float tx = s[3] - (by * s[2] - bz * s[1]);             // torque about b = M_t - (b - t) x F
        const float ty = s[4] - (bz * s[0] - bx * s[2]);
        const float tz = s[5] - (bx * s[1] - by * s[0]);
        gth = wx * tx + wy * ty + wz * tz;
    }
}

// ------------------------------------------------------------------ a3..a6: one pose evaluation by the whole CTA
// In : t[3], unit q[4] (uniform), theta (lane g holds the torsion angle of fragment g).
// Out: ENERGY: e_inter, e_intra (uniform over the CTA); GRAD: g6 = {dE/dt, dE/domega about t} (uniform), gth = dE/dtheta
//      on lane g (O9); x, y, z = this thread's atom (valid when `active`).
// MDN: the mixture-density term (mdn.cuh); the lanes of an atom share its residues (lane `part` takes residues part,
// part + lpa, ...), their shares join the pair force / the energy sums before the fixed-order reductions.
// DIRECT: the receptor term by direct pair sums over the receptor atoms (cta_rec_direct) instead of the grid lookup; the lanes
// of an atom share the atoms of every slice, their shares join the pair force.
template <bool GRAD, bool ENERGY, bool MDN, bool DIRECT>
__device__ __forceinline__ void cta_eval(const CtaTopo& S, const DGrid& G, const DParams& P, const PairK& K, const CtaFrag& F,
                                         const MdnDev& M, const float4* __restrict__ mdn_par, const RecDev& RD,
                                         int max_depth, const float t[3], const float q[4], float theta,
                                         int atom, int part, bool active, float& x, float& y, float& z,
                                         float& e_inter, float& e_intra, float g6[6], float& gth) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, n = S.n;

    float R[9], p[3];
    cta_frames(F, max_depth, t, q, theta, R, p);
    // this thread's atom: x_a = R_frag(a) r_a + p_frag(a); the group's first lane publishes it and starts the gathers
    const int m = active ? S.meta[atom] : 0;
    {
        const int fr = (m >> 8) & 0xff;
        float A[9], b[3];
#pragma unroll
        for (int i = 0; i < 9; ++i) A[i] = __shfl_sync(FULL_MASK, R[i], fr);
#pragma unroll
        for (int i = 0; i < 3; ++i) b[i] = __shfl_sync(FULL_MASK, p[i], fr);
        const float4 r = S.ref[active ? atom : 0];
        x = A[0] * r.x + A[1] * r.y + A[2] * r.z + b[0];
        y = A[3] * r.x + A[4] * r.y + A[5] * r.z + b[1];
        z = A[6] * r.x + A[7] * r.y + A[8] * r.z + b[2];
    }
    const bool lead = active && part == 0;
    GridCell cell;
    float4 glo = make_float4(0.f, 0.f, 0.f, 0.f), ghi = glo;
    if (lead) {
        S.X[atom] = x; S.X[n + atom] = y; S.X[2 * n + atom] = z;
        if (!DIRECT) {
            cell = grid_locate(G, m & 0xff, x, y, z);
            glo = __ldg(cell.p); ghi = __ldg(cell.p + 1);
        }
    }
    __syncthreads();

    // ---- a5 intra-ligand pairs (O6)
    float eL = 0.f, eC = 0.f, eH = 0.f, fx = 0.f, fy = 0.f, fz = 0.f;
    if (GRAD) {
        if (active) {
            const int k1 = S.rows[atom + 1];
            for (int k = S.rows[atom] + part; k < k1; k += 4 * S.lpa) {
                float dx[4], dy[4], dz[4], c[4];
                bool hb[4], ok[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int kk = k + u * S.lpa;
                    ok[u] = kk < k1;
                    const uint2 rec = S.recs[ok[u] ? kk : k];
                    const int b = (int)(rec.x & 0xffu);
                    dx[u] = x - S.X[b]; dy[u] = y - S.X[n + b]; dz[u] = z - S.X[2 * n + b];
                    c[u] = __uint_as_float(rec.y); hb[u] = (rec.x >> 8) & 1u;
                }
                cta_pairs4<true, ENERGY>(K, dx, dy, dz, c, hb, ok, eL, eC, eH, fx, fy, fz);
            }
        }
        eL *= 0.5f; eC *= 0.5f; eH *= 0.5f;                         // every pair was visited from both ends
    } else {
        const uint2* flat = S.flat;
        float f0 = 0.f, f1 = 0.f, f2 = 0.f;
        const int nt = (int)blockDim.x;
        for (int k = tid; k < S.P; k += 4 * nt) {
            float dx[4], dy[4], dz[4], c[4];
            bool hb[4], ok[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int kk = k + u * nt;
                ok[u] = kk < S.P;
                const uint2 rec = flat[ok[u] ? kk : k];
                const int a = (int)(rec.x & 0xffu), b = (int)((rec.x >> 8) & 0xffu);
                dx[u] = S.X[a] - S.X[b]; dy[u] = S.X[n + a] - S.X[n + b]; dz[u] = S.X[2 * n + a] - S.X[2 * n + b];
                c[u] = __uint_as_float(rec.y); hb[u] = (rec.x >> 16) & 1u;
            }
            cta_pairs4<false, true>(K, dx, dy, dz, c, hb, ok, eL, eC, eH, f0, f1, f2);
        }
    }
    // ---- a4 receptor term of this thread's atom (the gathers were issued before the barrier)
    float ei = 0.f, gx = 0.f, gy = 0.f, gz = 0.f;
    if (!DIRECT && lead) ei = grid_blend<GRAD>(G, P.k_wall, cell, glo, ghi, gx, gy, gz);
    if (DIRECT) cta_rec_direct<GRAD, ENERGY>(RD, K, active, m & 0xff, x, y, z, part, S.lpa, ei, fx, fy, fz);
    if (MDN && active) {
        float mx = 0.f, my = 0.f, mz = 0.f;
        mdn_atom_shared(M, mdn_par, n, atom, x, y, z, part, S.lpa, GRAD, ei, mx, my, mz);   // the atom's lanes split its candidate runs
        if (GRAD) { fx = fmaf(mx, K.inv_kappa, fx); fy = fmaf(my, K.inv_kappa, fy); fz = fmaf(mz, K.inv_kappa, fz); }   // kappa units, like the pair force
    }
    if (GRAD) {
        for (int o = S.lpa >> 1; o > 0; o >>= 1) {                  // the atom's lanes are adjacent: fixed-order tree
            fx += __shfl_xor_sync(FULL_MASK, fx, o);
            fy += __shfl_xor_sync(FULL_MASK, fy, o);
            fz += __shfl_xor_sync(FULL_MASK, fz, o);
        }
        if (lead) {
            const float Fx = fmaf(K.kappa, fx, gx), Fy = fmaf(K.kappa, fy, gy), Fz = fmaf(K.kappa, fz, gz);
            const float ax = x - t[0], ay = y - t[1], az = z - t[2];
            float4* af = reinterpret_cast<float4*>(S.AF) + 2 * atom;
            af[0] = make_float4(Fx, Fy, Fz, 0.f);
            af[1] = make_float4(ay * Fz - az * Fy, az * Fx - ax * Fz, ax * Fy - ay * Fx, 0.f);
        }
    }
    if (ENERGY) {
        const float ea = fmaf(K.w_clash_ln2, eC, -fmaf(K.w_long, eL, K.w_hbond * eH));
        const float si = warp_sum(ei), sa = warp_sum(ea);
        if (lane == 0) { S.red[2 * warp] = si; S.red[2 * warp + 1] = sa; }
    }
    __syncthreads();
    if (ENERGY) {
        e_inter = 0.f; e_intra = 0.f;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { e_inter += S.red[2 * w]; e_intra += S.red[2 * w + 1]; }
    }
    if (!GRAD) return;

    cta_reverse(S, F, R, p, t, g6, gth);
}

// ------------------------------------------------------------------ a3..a6 for ligands above 64 atoms: dense partner sweep
// The same contract as cta_eval, for a CTA of NW warps (4: score kernel, one atom per thread; 2: MC kernel, two atoms per thread).
// Sweep (internal.h): this warp's lanes hold the atoms l = c0 + lane of one 32-atom chunk after another and meet the partners
// b = b0 + 4 * warp + u, u = 0..3 (warp-uniform: one broadcast 16-byte load each); the other warps take the other partners, so a
// chunk's force is the sum of the warps' partials -- fixed order, after a barrier.  GRAD: all partners (both ends of every
// pair); energy only: the partners b > l.  A last chunk of at most 16 atoms is held twice, by the two half-warps, which split
// the partners between them.  x0, y0, z0: the coordinates of atom threadIdx.x.
template <bool GRAD, bool ENERGY, bool MDN, bool DIRECT, int NW>
__device__ __forceinline__ void cta_eval_dense(const CtaTopo& S, const DGrid& G, const DParams& P, const PairK& K, const CtaFrag& F,
                                               const MdnDev& M, const float4* __restrict__ mdn_par, const RecDev& RD,
                                               int max_depth, const float t[3], const float q[4], float theta,
                                               float& x0, float& y0, float& z0,
                                               float& e_inter, float& e_intra, float g6[6], float& gth) {
    constexpr int APT = TRIDSK_CTA_WARPS / NW;                      // atoms per thread: 128 atoms at most
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, n = S.n;
    float R[9], p[3];
    cta_frames(F, max_depth, t, q, theta, R, p);

    // this thread's atoms: x_a = R_frag(a) r_a + p_frag(a), published with the atom type; the gathers start
    float x[APT], y[APT], z[APT];
    int m[APT];
    bool act[APT];
    GridCell cell[APT];
    float4 glo[APT], ghi[APT];
#pragma unroll
    for (int k = 0; k < APT; ++k) {
        const int atom = tid + 32 * NW * k;
        act[k] = atom < n;
        m[k] = act[k] ? S.meta[atom] : 0;
        const int fr = (m[k] >> 8) & 0xff;
        float A[9], b[3];
#pragma unroll
        for (int i = 0; i < 9; ++i) A[i] = __shfl_sync(FULL_MASK, R[i], fr);
#pragma unroll
        for (int i = 0; i < 3; ++i) b[i] = __shfl_sync(FULL_MASK, p[i], fr);
        const float4 r = S.ref[act[k] ? atom : 0];
        x[k] = A[0] * r.x + A[1] * r.y + A[2] * r.z + b[0];
        y[k] = A[3] * r.x + A[4] * r.y + A[5] * r.z + b[1];
        z[k] = A[6] * r.x + A[7] * r.y + A[8] * r.z + b[2];
        glo[k] = make_float4(0.f, 0.f, 0.f, 0.f); ghi[k] = glo[k];
        if (act[k]) {
            S.X4[atom] = make_float4(x[k], y[k], z[k], __int_as_float(m[k] & 0xff));
            if (!DIRECT) {
                cell[k] = grid_locate(G, m[k] & 0xff, x[k], y[k], z[k]);
                glo[k] = __ldg(cell[k].p); ghi[k] = __ldg(cell[k].p + 1);
            }
        }
    }
    x0 = x[0]; y0 = y[0]; z0 = z[0];
    __syncthreads();

    // ---- a5 intra-ligand pairs (O6)
    float eL = 0.f, eC = 0.f, eH = 0.f;
    const int npad = S.npad, plane = (npad >> 5) * npad;
    float4* part = S.part + warp * npad;
    for (int c0 = 0; c0 < npad; c0 += 32) {
        const bool half = GRAD && n - c0 <= 16;
        const int l = c0 + (half ? (lane & 15) : lane), bo = half ? (lane >> 4) << 2 : 0, per = half ? 8 : 4;
        const unsigned lbit = 1u << (l & 31);
        const float4 me = S.X4[l];
        const float* trow = S.tt + 33 * __float_as_int(me.w);
        const unsigned* irow = S.msk + (GRAD ? 0 : 2 * plane) + (c0 >> 5) * npad;
        const unsigned* hrow = irow + plane;
        float ax = 0.f, ay = 0.f, az = 0.f;
        for (int bb = (GRAD ? 0 : c0) + per * warp; bb < n; bb += per * NW) {
            const int b0 = bb + bo;
            const uint4 iw = *reinterpret_cast<const uint4*>(irow + b0);
            const uint4 hw = *reinterpret_cast<const uint4*>(hrow + b0);
            const unsigned in[4] = {iw.x, iw.y, iw.z, iw.w};
            float4 pb[4];
            float c[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                pb[u] = S.X4[b0 + u];
                c[u] = trow[__float_as_int(pb[u].w)];
                c[u] = (in[u] & lbit) ? c[u] : -1e15f;
            }
            cta_dense4<GRAD, ENERGY>(K, me, pb, c, hw, lbit, eL, eC, eH, ax, ay, az);
        }
        if (GRAD) {
            if (half) {
                ax += __shfl_xor_sync(FULL_MASK, ax, 16); ay += __shfl_xor_sync(FULL_MASK, ay, 16); az += __shfl_xor_sync(FULL_MASK, az, 16);
            }
            part[l] = make_float4(ax, ay, az, 0.f);
        }
    }
    if (GRAD) {
        eL *= 0.5f; eC *= 0.5f; eH *= 0.5f;                         // every pair was visited from both ends
        __syncthreads();
    }

    // ---- a4 receptor term of this thread's atoms (the gathers were issued before the first barrier), force and moment records
    float ei = 0.f;
#pragma unroll
    for (int k = 0; k < APT; ++k) {
        const int atom = tid + 32 * NW * k;
        float gx = 0.f, gy = 0.f, gz = 0.f, fx = 0.f, fy = 0.f, fz = 0.f;
        if (DIRECT) cta_rec_direct<GRAD, ENERGY>(RD, K, act[k], m[k] & 0xff, x[k], y[k], z[k], 0, 1, ei, fx, fy, fz);   // (the whole warp calls)
        if (act[k]) {
            if (!DIRECT) ei += grid_blend<GRAD>(G, P.k_wall, cell[k], glo[k], ghi[k], gx, gy, gz);
            if (GRAD) {
#pragma unroll
                for (int w = 0; w < NW; ++w) { const float4 f = S.part[w * npad + atom]; fx += f.x; fy += f.y; fz += f.z; }
            }
            if (MDN) {
                float mx = 0.f, my = 0.f, mz = 0.f;
                mdn_atom(M, mdn_par, n, atom, x[k], y[k], z[k], 0, 1, GRAD, ei, mx, my, mz);
                if (GRAD) { fx = fmaf(mx, K.inv_kappa, fx); fy = fmaf(my, K.inv_kappa, fy); fz = fmaf(mz, K.inv_kappa, fz); }
            }
            if (GRAD) {
                const float Fx = fmaf(K.kappa, fx, gx), Fy = fmaf(K.kappa, fy, gy), Fz = fmaf(K.kappa, fz, gz);
                const float rx = x[k] - t[0], ry = y[k] - t[1], rz = z[k] - t[2];
                float4* af = reinterpret_cast<float4*>(S.AF) + 2 * atom;
                af[0] = make_float4(Fx, Fy, Fz, 0.f);
                af[1] = make_float4(ry * Fz - rz * Fy, rz * Fx - rx * Fz, rx * Fy - ry * Fx, 0.f);
            }
        }
    }
    if (ENERGY) {
        const float ea = fmaf(K.w_clash_ln2, eC, -fmaf(K.w_long, eL, K.w_hbond * eH));
        const float si = warp_sum(ei), sa = warp_sum(ea);
        if (lane == 0) { S.red[2 * warp] = si; S.red[2 * warp + 1] = sa; }
    }
    __syncthreads();
    if (ENERGY) {
        e_inter = 0.f; e_intra = 0.f;
#pragma unroll
        for (int w = 0; w < NW; ++w) { e_inter += S.red[2 * w]; e_intra += S.red[2 * w + 1]; }
    }
    if (!GRAD) return;
    cta_reverse(S, F, R, p, t, g6, gth);
}

// ROUNDS: 0 = pair records (ligands of up to 64 atoms, 128 threads), 1 = dense partner sweep with two warps per chain (MC kernel),
// 2 = decided at run time by S.rounds, 128 threads (score kernel).
template <bool GRAD, bool ENERGY, bool MDN, int ROUNDS, bool DIRECT>
__device__ __forceinline__ void cta_eval_any(const CtaTopo& S, const DGrid& G, const DParams& P, const PairK& K, const CtaFrag& F,
                                             const MdnDev& M, const float4* __restrict__ mdn_par, const RecDev& RD,
                                             int max_depth, const float t[3], const float q[4], float theta,
                                             int atom, int part, bool active, float& x, float& y, float& z,
                                             float& e_inter, float& e_intra, float g6[6], float& gth) {
    if constexpr (ROUNDS == 1) {
        cta_eval_dense<GRAD, ENERGY, MDN, DIRECT, 2>(S, G, P, K, F, M, mdn_par, RD, max_depth, t, q, theta, x, y, z, e_inter, e_intra, g6, gth);
    } else {
        if (ROUNDS == 2 && S.rounds)
            cta_eval_dense<GRAD, ENERGY, MDN, DIRECT, 4>(S, G, P, K, F, M, mdn_par, RD, max_depth, t, q, theta, x, y, z, e_inter, e_intra, g6, gth);
        else
            cta_eval<GRAD, ENERGY, MDN, DIRECT>(S, G, P, K, F, M, mdn_par, RD, max_depth, t, q, theta, atom, part, active, x, y, z, e_inter, e_intra, g6, gth);
    }
}

// ------------------------------------------------------------------ chain state I/O: lane g <-> pose[7 + tor(g)]
__device__ __forceinline__ void cta_load_pose(const float* __restrict__ src, const CtaFrag& F, float t[3], float q[4], float& th) {
    t[0] = src[0]; t[1] = src[1]; t[2] = src[2];
    q[0] = src[3]; q[1] = src[4]; q[2] = src[5]; q[3] = src[6];
    th = F.tor >= 0 ? src[7 + F.tor] : 0.f;
}
__device__ __forceinline__ void cta_store_pose(float* __restrict__ dst, const CtaFrag& F, int T, int stride, const float t[3],
                                               const float q[4], float th) {
    const int lane = threadIdx.x & 31;
    if (lane == 0) {
        dst[0] = t[0]; dst[1] = t[1]; dst[2] = t[2];
        dst[3] = q[0]; dst[4] = q[1]; dst[5] = q[2]; dst[6] = q[3];
    }
    if (F.tor >= 0) dst[7 + F.tor] = th;
    for (int e = 7 + T + lane; e < stride; e += 32) dst[e] = 0.f;
}

// ------------------------------------------------------------------ the fused MC kernel, one CTA per chain
// Record instance: 128 threads, registers for 3 resident CTAs per SM (with 4 x 128 registers, C2 goes 6.0 -> 6.3 ms).  Dense
// instance: 64 threads and 128 registers, EIGHT chains resident per SM (with the mixture-density term: 255 registers, four chains --
// an 80-atom dock under the full score 490 -> 345 ms; the record instance with the term is faster at 168 than at 255: 60.5 / 71.3 ms).
// DIRECT: the receptor term by direct pair sums (tridsk_dock_opts.receptor_direct), without the mixture-density term.
template <bool MDN, int ROUNDS, bool DIRECT>
__global__ void __launch_bounds__(ROUNDS ? 64 : 128, ROUNDS ? (MDN ? 4 : 8) : 3) mc_cta_kernel(const McLaunch a) {
    extern __shared__ __align__(16) unsigned char cta_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lig = a.lig_list[blockIdx.x / a.n_chains];
    const int chain = blockIdx.x % a.n_chains;
    const LigHdr* h = a.hdr + lig;
    CtaTopo S;
    CtaFrag F;
    cta_stage(S, F, cta_smem, h, a.atom_f4, a.atom_i, a.lane_frags, a.cta_rows, a.cta_recs, a.cta_rtab, a.P, a.cta_dense_n);
    const DParams& P = a.P;
    const PairK K = make_pairk(P);
    const float4* mdn_par = MDN ? a.mdn.par + a.mdn.lig_off[lig] : nullptr;
    const int T = S.T, max_depth = h->max_depth;
    const int atom = tid / S.lpa, part = tid % S.lpa;
    const bool active = atom < S.n;
    const size_t cidx = (size_t)lig * a.n_chains + chain;
    const uint2 key = make_uint2((uint32_t)a.seed, (uint32_t)(a.seed >> 32));
    const uint32_t gchain = (uint32_t)(a.chain_base + chain);

    float ct[3], cq[4], cth, ecur;          // current accepted state (every warp holds a copy)
    float bt[3], bq[4], bth, ebest;         // best state seen
    float x, y, z, g6[6], gth, ei, ea;

    if (a.init_mode == 2) {                 // resume
        cta_load_pose(a.pose_cur + cidx * a.pose_stride, F, ct, cq, cth);
        cta_load_pose(a.pose_best + cidx * a.pose_stride, F, bt, bq, bth);
        ecur = a.e_cur[cidx]; ebest = a.e_best[cidx];
    } else {
        if (a.init_mode == 1) {
            cta_load_pose(a.init_poses + cidx * a.pose_stride, F, ct, cq, cth);
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
            // torsion k takes element k % 4 of block 4 + k / 4, i.e. of lane 2 + k / 4
            const int k = F.tor >= 0 ? F.tor : 0, src = 2 + (k >> 2);
            const float v0 = __shfl_sync(FULL_MASK, u0, src & 31), v1 = __shfl_sync(FULL_MASK, u1, src & 31);
            const float v2 = __shfl_sync(FULL_MASK, u2, src & 31), v3 = __shfl_sync(FULL_MASK, u3, src & 31);
            const float uu = (k & 3) == 0 ? v0 : (k & 3) == 1 ? v1 : (k & 3) == 2 ? v2 : v3;
            cth = F.tor >= 0 ? PI_F * (2.f * uu - 1.f) : 0.f;
        }
        cta_eval_any<false, true, MDN, ROUNDS, DIRECT>(S, a.grid, P, K, F, a.mdn, mdn_par, a.rec, max_depth, ct, cq, cth, atom, part, active, x, y, z, ei, ea, g6, gth);
        ecur = ei + ea;
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
        } else if (F.tor == entity - 2) {
            pth = PI_F * (2.f * u1 - 1.f);
        }

        // a3..a7: n_refine Adam steps on the 6+T tangent components (moments reset every MC step, G12)
        float m[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, v[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        float b1p = 1.f, b2p = 1.f;
        for (int rf = 0; rf < P.n_refine; ++rf) {
            cta_eval_any<true, false, MDN, ROUNDS, DIRECT>(S, a.grid, P, K, F, a.mdn, mdn_par, a.rec, max_depth, pt, pq, pth, atom, part, active, x, y, z, ei, ea, g6, gth);
            b1p *= P.adam_b1; b2p *= P.adam_b2;
            const float c1 = __fdividef(1.f, 1.f - b1p), c2 = __fdividef(1.f, 1.f - b2p);
            float g[7] = {g6[0], g6[1], g6[2], g6[3], g6[4], g6[5], gth}, dl[7];
#pragma unroll
            for (int i = 0; i < 7; ++i) {                            // division / square root to 2 ulp: far inside the tolerance
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
            pth = F.tor >= 0 ? th : 0.f;
        }

        // a8: energy of the refined proposal, Metropolis, best tracking
        cta_eval_any<false, true, MDN, ROUNDS, DIRECT>(S, a.grid, P, K, F, a.mdn, mdn_par, a.rec, max_depth, pt, pq, pth, atom, part, active, x, y, z, ei, ea, g6, gth);
        const float enew = ei + ea;
        const bool accept = isfinite(enew) && (um < expf(-P.beta * (enew - ecur)));
        if (a.trace != nullptr && tid == 0) {
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

    if (warp == 0) {
        cta_store_pose(a.pose_cur + cidx * a.pose_stride, F, T, a.pose_stride, ct, cq, cth);
        cta_store_pose(a.pose_best + cidx * a.pose_stride, F, T, a.pose_stride, bt, bq, bth);
        if (lane == 0) { a.e_cur[cidx] = ecur; a.e_best[cidx] = ebest; }
    }
}

// ------------------------------------------------------------------ tridsk_score_grad, CTA form: one CTA per pose
template <bool MDN>
__global__ void __launch_bounds__(128) score_cta_kernel(const ScoreLaunch a) {
    extern __shared__ __align__(16) unsigned char cta_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i = blockIdx.x;
    const int lig = a.lig_index[i];
    const LigHdr* h = a.hdr + lig;
    CtaTopo S;
    CtaFrag F;
    cta_stage(S, F, cta_smem, h, a.atom_f4, a.atom_i, a.lane_frags, a.cta_rows, a.cta_recs, a.cta_rtab, a.P, TRIDSK_CTA_ROUNDS_N);
    const PairK K = make_pairk(a.P);
    const float4* mdn_par = MDN ? a.mdn.par + a.mdn.lig_off[lig] : nullptr;
    const int atom = tid / S.lpa, part = tid % S.lpa;
    const bool active = atom < S.n;
    float t[3], q[4], th, x, y, z, g6[6], gth = 0.f, ei, ea;
    RecDev no_rec;
    no_rec.atoms = nullptr;
    cta_load_pose(a.poses + (size_t)i * a.pose_stride, F, t, q, th);
    quat_normalise(q);
    if (a.grad != nullptr) cta_eval_any<true, true, MDN, 2, false>(S, a.grid, a.P, K, F, a.mdn, mdn_par, no_rec, h->max_depth, t, q, th, atom, part, active, x, y, z, ei, ea, g6, gth);
    else cta_eval_any<false, true, MDN, 2, false>(S, a.grid, a.P, K, F, a.mdn, mdn_par, no_rec, h->max_depth, t, q, th, atom, part, active, x, y, z, ei, ea, g6, gth);
    if (tid == 0) { a.energy[3 * (size_t)i] = ei + ea; a.energy[3 * (size_t)i + 1] = ei; a.energy[3 * (size_t)i + 2] = ea; }
    if (a.grad != nullptr && warp == 0) {
        float* g = a.grad + (size_t)i * a.grad_stride;
        if (lane == 0) { g[0] = g6[0]; g[1] = g6[1]; g[2] = g6[2]; g[3] = g6[3]; g[4] = g6[4]; g[5] = g6[5]; }
        if (F.tor >= 0) g[6 + F.tor] = gth;
        for (int e = 6 + S.T + lane; e < a.grad_stride; e += 32) g[e] = 0.f;
    }
    if (a.coords != nullptr) {
        float* c = a.coords + (size_t)i * a.coord_stride * 3;
        if (active && part == 0) {
            const int orig = (S.meta[atom] >> 16) & 0xff;
            c[3 * orig] = x; c[3 * orig + 1] = y; c[3 * orig + 2] = z;
        }
        for (int e = 3 * S.n + tid; e < 3 * a.coord_stride; e += blockDim.x) c[e] = 0.f;
    }
}

// per device (function attributes are per device): called by tridsk_create
cudaError_t mc_cta_prepare() {
    cudaError_t e = cudaFuncSetAttribute(mc_cta_kernel<false, 0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TRIDSK_SMEM_MAX_CTA);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mc_cta_kernel<true, 0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TRIDSK_SMEM_MAX_CTA);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mc_cta_kernel<false, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TRIDSK_SMEM_MAX_CTA);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mc_cta_kernel<true, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TRIDSK_SMEM_MAX_CTA);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mc_cta_kernel<false, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, TRIDSK_SMEM_MAX_CTA);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(mc_cta_kernel<false, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, TRIDSK_SMEM_MAX_CTA);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(score_cta_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TRIDSK_SMEM_MAX_CTA);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(score_cta_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, TRIDSK_SMEM_MAX_CTA);
    return e;
}

cudaError_t launch_mc_cta(cudaStream_t s, const McLaunch& a, int rounds, size_t smem_bytes) {
    const long long blocks = (long long)a.n_list * a.n_chains;
    if (blocks <= 0) return cudaSuccess;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    const unsigned nb = (unsigned)blocks;
    if (a.rec.atoms) {                                            // direct receptor sums (the host does not pair them with E_MDN)
        if (a.mdn.n_res > 0) return cudaErrorInvalidValue;
        if (rounds) mc_cta_kernel<false, 1, true><<<nb, 64, smem_bytes, s>>>(a); else mc_cta_kernel<false, 0, true><<<nb, 128, smem_bytes, s>>>(a);
    } else if (a.mdn.n_res > 0) {
        if (rounds) mc_cta_kernel<true, 1, false><<<nb, 64, smem_bytes, s>>>(a); else mc_cta_kernel<true, 0, false><<<nb, 128, smem_bytes, s>>>(a);
    } else {
        if (rounds) mc_cta_kernel<false, 1, false><<<nb, 64, smem_bytes, s>>>(a); else mc_cta_kernel<false, 0, false><<<nb, 128, smem_bytes, s>>>(a);
    }
    return cudaGetLastError();
}

cudaError_t launch_score_cta(cudaStream_t s, const ScoreLaunch& a, size_t smem_bytes) {
    if (a.n_pose <= 0) return cudaSuccess;
    if (a.mdn.n_res > 0) score_cta_kernel<true><<<a.n_pose, 128, smem_bytes, s>>>(a);
    else score_cta_kernel<false><<<a.n_pose, 128, smem_bytes, s>>>(a);
    return cudaGetLastError();
}
