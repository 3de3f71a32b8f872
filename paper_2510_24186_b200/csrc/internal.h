// internal.h -- structures shared by the translation units of libtridsk (host + device).
// Nothing here is visible through the C-ABI (include/tridsk.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <memory>
#include <string>
#include <vector>

#include "../../include/tridsk.h"

#define TRIDSK_WARPS_PER_CTA 4
#define TRIDSK_MAX_J 4           // atoms per lane (n_atoms <= 32 * MAX_J)
#define TRIDSK_MAX_TILES 10      // J(J+1)/2 tiles of the pair schedule
#define TRIDSK_CTA_MAX_LIG 1024  // batches up to this size also carry the CTA-per-chain pair format
#define TRIDSK_SCRATCH 12       // scratch buffers owned by a ctx (api.cu names the slots)
#define TRIDSK_BRANCHES 16       // parallel branches of a dock's launch series (ctx stream + side streams)

// ---------------------------------------------------------------- device-side packed formats
// Scoring / sampling constants in the form the kernels use (fp32).
struct DParams {
    float w_long, w_clash, w_hbond;
    float long_mu, long_inv_two_sigma2, long_dmax;
    float hb_mu, hb_inv_two_sigma2, hb_dmax, hb_dclash;
    float d_floor, k_wall;
    float beta, lr, adam_b1, adam_b2, adam_eps;
    float pert_trans, pert_rot, w_tor;
    int n_refine;
};

// Receptor grid: fp32 planes [type][z][y][x] (x fastest).
struct DGrid {
    const float* g;
    const float4* gp;             // cell-packed copy, 32 bytes per node: gp[2 * node] = {g(x,y), g(x+1,y), g(x,y+1), g(x+1,y+1)} at z, gp[2 * node + 1]
                                  // = the same at z + 1 (edges clamped): the 8 corners of the trilinear cell based at the node in one sector
    int nx, ny, nz, n_types;
    size_t plane;                 // nx*ny*nz
    float ox, oy, oz, h, inv_h;
};

// The mixture-density term (mdn.cuh, O15) attached to a ligand batch; n_res == 0: absent.
// Parameters: a (residue, atom) pair owns a SLOT of blocks; a block holds up to ten components as {a, mu, nk2} x 10 (30 floats
// + 2 unused = 128 bytes); the last block is cut to whole 32-byte chunks.  K = 10: one 128-byte cache line per pair.
__host__ __device__ static inline int mdn_slot_f4(int K) {          // float4 units per slot
    const int nb = (K + 9) / 10, kl = K - 10 * (nb - 1);
    return 2 * (4 * (nb - 1) + (3 * kl + 7) / 8);
}
struct MdnDev {
    int n_res, K, K4;             // K4 = mdn_slot_f4(K): float4 units per (residue, atom) slot in par
    const float4* sph;            // [n_res] bounding sphere of a residue: centre, (radius + d_cut)^2
    const int* res_off;           // [n_res + 1] into rec
    const float4* rec;            // residue atoms {x, y, z, 0}
    const float4* par;            // packed parameter slots, ligand-major, [n_res][n][K4] per ligand, INTERNAL atom order
    const long long* lig_off;     // [n_lig] start of a ligand's block in par (float4 units)
    float d_cut;
    // cell list: a uniform grid over the residues' bounding box grown by d_cut; cell c holds, as ONE contiguous stream
    // sorted by (residue, atom index), every receptor atom {x, y, z, w} within d_cut + half a cell diagonal of the
    // cell's centre (runs padded to an even number of entries).  For a point of the cell, a residue's minimum over the listed atoms equals its true minimum distance
    // whenever that is below d_cut (the arg-min atom is then listed), and is >= d_cut otherwise.
    float glo[3], inv_cell;
    int nc[3];
    const int* cell_off;          // [ncells + 1]
    const float4* cell_at;
    // run directory (for the mapping whose lanes SHARE an atom's candidate runs): the runs of cell c are dir[dir_off[c] .. dir_off[c + 1]),
    // each {header = residue id | run length << 16, position of the run in cell_at}
    const int* dir_off;           // [ncells + 1]
    const int2* dir;
};

// Direct-pair receptor mode: the receptor atoms sorted into cubic cells of edge = the pair function's
// range; atoms == nullptr: the receptor term comes from the grid.
struct RecDev {
    const float4* atoms;          // {x, y, z, type bits}, sorted by cell, input order inside a cell
    const int* cell_off;          // [ncells + 1]
    const float* radius;          // [n_types]
    const unsigned char* role;    // [n_types]
    int nc[3], span;              // cells per axis; the cut-off spans `span` cells
    float lo[3], inv_cell, cell, cut2;
};

// Per-ligand header.  Atoms are stored in an INTERNAL order (depth-first over the torsion tree) so that
// the atoms of every torsion's subtree are one contiguous index range; lane l of a chain's warp owns
// atoms a = j*S + l, j < J ("stripes").
struct LigHdr {
    int n, T, J, S;
    int atom_off;                 // into atom_f4 / atom_i
    int frag_off;                 // into frags (T+1 records)
    int round_off;                // into rounds
    int max_depth;
    int tile_off[TRIDSK_MAX_TILES + 1];   // round ranges per (j1<=j2) tile, relative to round_off
    int n_pairs;
    int ls_off;                   // lane format: into lane_stream (ls_len 16-byte header units, see LaneFrag)
    int ls_len;
    int rec_off;                  // lane format: into lane_recs (n_rec records, in the order the stream consumes them)
    int n_rec;
    int cta_row_off;              // CTA format: into cta_rows (n + 1 row offsets, relative to the ligand's records)
    int cta_rec_off;              // CTA format: into cta_recs (2 n_pairs row records, then n_pairs flat records)
    int cta_rt_off;               // CTA format, n > 64: into cta_rtab ((n / 2) * n entries of the round table); -1: none
};

// Lane format (mc_lane.cu).  Fragments are re-indexed in depth-first PRE-order g = 0..T (0 = root), so that the
// subtree of g is the contiguous fragment range [g, g_end) and a fragment at depth d finds its parent's frame in
// frame slot d - 1.  One record per fragment:
struct LaneFrag {
    float ux, uy, uz;             // torsion axis (unit) and axis point (atom b_k), reference frame
    float ox, oy, oz;
    int lo, own_hi;               // the fragment's own atoms [lo, own_hi), internal order
    int parent;                   // pre-order index of the parent fragment (0 for the root)
    int depth;                    // root = 0
    int axis;                     // internal indices of the axis atoms a_k | b_k << 8
    int tor;                      // torsion index k of the pose vector (pose[7 + k]); -1 for the root
};
// The intra-ligand pair set as a uniform instruction stream: 16-byte header units + a record array that the headers
// consume in order.  For every fragment g (pre-order):
//   {n_tiles, 0, 0, 0}
//   per tile (1..4 consecutive own atoms a0 .. a0+w-1 of g):   {a0, w, n_runs, 0}
//     per run (partner atoms in ONE other fragment fb):          {fb, n_rec, 0, 0}   -> the next n_rec records
// Of the two fragments of a pair, the one that needs fewer records supplies the tiles (api.cu).
// One record = one partner atom b against the 4 slots of the tile.  In global memory (LaneRec) it holds what depends
// on the ligand only; lane_stage turns it into the 20-byte shared-memory form (two arrays) that also depends on the
// parameters:  c[4] = dvdw + long_mu (slot without a pair -- excluded, or beyond the tile width: -1e15), and one word
// scale * b | hbmask << 16 (scale * b = where atom b's coordinates start in the chain's coordinate store).  The pair arithmetic then has no topology branch: a slot without a pair evaluates to exactly
// zero (its clash distance c - mu is negative).
struct LaneRec {
    float dvdw[4];                // r_a + r_b per slot; < 0 for a slot without a pair
    uint32_t b, hbmask;           // partner atom (internal index); bit i: slot i is a donor/acceptor pair
    uint32_t pad[2];
};
#define TRIDSK_LANE_REC_SMEM 20

// CTA format (mc_cta.cu): the pair set twice over.  Row form, for the gradient: for every atom a (internal order) the
// partners b of a, {b | hb << 8, dvdw bits}, rows delimited by cta_rows -- every pair appears in both rows, so an atom's
// force is a sum its own threads own (no scatter, no atomics).  Flat form, for energy-only evaluations: every pair once,
// {a | b << 8 | hb << 16, dvdw bits}, sorted by (a, b).  Fragments are the LaneFrag records (pre-order).

// Ligands of more than 64 atoms use a DENSE PARTNER SWEEP instead of pair records: a warp takes 32 consecutive atoms l (one
// per lane) and sweeps the partner b over the ligand, four partners in flight; the partner's coordinates and atom type are ONE
// broadcast 16-byte shared-memory load, c = dvdw + mu comes from a (type, type) table in shared memory (row stride 33: the
// lanes' rows fall into different banks), and whether (l, b) is in the pair set / is a donor-acceptor pair from 32-bit lane
// masks per (b, 32-atom chunk): a visit outside the pair set gets c = -1e15 and adds exactly zero, and the hydrogen-bond term
// is skipped, warp-uniformly, for the partners that have no such pair.  Gradient evaluations visit every pair from both ends
// (an atom's force is a sum its own lane owns: no scatter, no atomics, bit-reproducible); energy-only evaluations visit the
// pairs l < b only (a second set of masks).  The masks are built in shared memory from the ROUND TABLE
// cta_rtab[(k - 1) * n + l], k = 1 .. n/2: the dvdw of pair (l, (l + k) mod n) as a float whose lowest mantissa bit is the
// donor/acceptor flag, or -1 if the pair is not in the set (for even n the items l >= n/2 of round n/2 repeat pairs and are
// absent).  The MC kernel gives such a chain TWO warps (64-thread CTAs, two atoms per thread outside the sweep), so that eight
// chains stay resident per SM.
#define TRIDSK_CTA_ROUNDS_N 64         // ligands above this many atoms always use the dense partner sweep (two warps per chain)
#define TRIDSK_CTA_DENSE_MIN 32        // ... and those above this many when the dock has more chains than the SMs hold at once (throughput
                                       // over latency: 48 atoms, 4 x 384 chains 13.3 -> 11.2 ms, but one dock of 64 atoms 4.5 -> 7.3 ms)

// Per-fragment record; fragment 0 is the root, fragment k+1 hangs off torsion k.
struct FragRec {
    float ux, uy, uz, ox;         // axis unit vector and axis point (atom b_k), reference frame
    float oy, oz;
    int own_hi;                   // the fragment's own atoms are [lo, own_hi) (internal order)
    int axis;                     // internal indices of the axis atoms: a_k | b_k << 8 (0 for the root)
    int parent, depth, lo, hi;    // parent fragment, depth (root = 0), subtree atom range [lo, hi)
};

// One round of the conflict-free pair schedule: in round (j1, j2, k) lane l evaluates the pair
// (atom j1*S + l, atom j2*S + (l+k) mod S) if bit l of `mask` is set; `hb` marks donor/acceptor pairs.
struct PairRound {
    uint32_t mask, hb;
    int k, pad;
};

struct McLaunch {
    // ligand batch
    const LigHdr* hdr;
    const float4* atom_f4;        // {ref x, y, z, vdW radius}
    const int* atom_i;            // type | frag << 8 | original index << 16
    const FragRec* frags;
    const PairRound* rounds;
    const LaneFrag* lane_frags;   // lane format: T + 1 records per ligand at frag_off, pre-order
    const uint4* lane_stream;     // lane format: the pair instruction stream (header units)
    const LaneRec* lane_recs;     // lane format: the pair records
    const int* cta_rows;          // CTA format
    const uint2* cta_recs;
    const float* cta_rtab;
    const int* lig_list;          // ligands handled by this launch (one bucket)
    int n_list;
    DGrid grid;
    DParams P;
    float box_min[3], box_max[3], centre[3], radius;
    int n_chains, pose_stride;
    int chain_base;               // global id of local chain 0 in the Philox counter (multi-GPU chain sharding)
    int lig_base;                 // global id of the handle's ligand 0 in the Philox counter (tridsk_screen docks a batch in two parts)
    int cta_dense_n;              // CTA kernel: ligands above this many atoms take the dense partner sweep
    unsigned long long seed;
    int first_step, n_steps;
    int init_mode;                // 0 Philox init, 1 from init_poses, 2 resume from state
    const float* init_poses;      // [n_lig][n_chains][pose_stride]
    float* pose_cur;              // [n_lig][n_chains][pose_stride]
    float* pose_best;
    float* e_cur;                 // [n_lig][n_chains]
    float* e_best;
    tridsk_trace_rec* trace;      // [n_lig][n_chains][trace_stride] or NULL
    int trace_stride, trace_off;
    int lane_region, tm_cols;     // tensor-memory lane kernel: shared-memory bytes per warp, TMEM columns per CTA
    int lane_minb;                // shared-memory lane kernel: register budget class (launch_bounds min blocks)
    MdnDev mdn;                   // n_res == 0: no mixture-density term
    RecDev rec;                   // atoms != nullptr: receptor term by direct pair sums (warp- and CTA-per-chain mappings)
};

struct ScoreLaunch {
    const LigHdr* hdr;
    const float4* atom_f4;
    const int* atom_i;
    const FragRec* frags;
    const PairRound* rounds;
    const LaneFrag* lane_frags;
    const uint4* lane_stream;
    const LaneRec* lane_recs;
    const int* cta_rows;
    const uint2* cta_recs;
    const float* cta_rtab;
    const int* seg_lig;           // lane score kernel: per CTA the ligand, and its poses perm[seg_start .. seg_start + seg_cnt)
    const int* seg_start;
    const int* seg_cnt;
    const int* perm;
    DGrid grid;
    DParams P;
    const int* lig_index;
    const float* poses;
    int n_pose, pose_stride;
    float* energy;                // [n_pose][3]
    float* grad; int grad_stride;
    float* coords; int coord_stride;
    MdnDev mdn;
};

struct TopkLaunch {
    const LigHdr* hdr;
    const float* e_best; const float* pose_best;
    int n_lig, n_chains, pose_stride, top_k;
    float w_tor;
    float* out_energy; float* out_pose; int* out_chain;
    // duplicate-removing form (cluster_rmsd > 0): the ligands' reference conformers and fragment records for the FK
    const float4* atom_f4; const LaneFrag* lane_frags;
    float cluster_rmsd;
    int max_atoms, max_tor;
};

// ---------------------------------------------------------------- lane-per-chain kernel: shared-memory budget
// One CTA = chains_per_cta chains of ONE ligand.  Shared memory = the ligand's topology (staged once per CTA)
// + per chain: coordinates X[3n], a scratch region that holds the fragment frames [12 max_depth] during the forward
// pass and the per-fragment wrenches [6(T+1)] during the reverse pass, current and proposed torsions [2T], and the
// torsion Adam moments [2T] when n_refine > 1.
#define TRIDSK_SMEM_PER_SM 233472      // 228 KB
#define TRIDSK_SMEM_RESERVED 1024      // per resident CTA
#define TRIDSK_SMEM_MAX_CTA 232448     // 227 KB opt-in maximum per CTA
__host__ __device__ static inline size_t lane_topo_bytes(int n, int T, int ls_len, int n_rec) {
    return 16 * (size_t)n + 16 * (size_t)((n + 3) / 4) + sizeof(LaneFrag) * (size_t)(T + 1) + 16 * (size_t)ls_len +
           (TRIDSK_LANE_REC_SMEM * (size_t)(n_rec + 1) + 15) / 16 * 16;   // + the pad record
}
__host__ __device__ static inline int lane_wslots(int T, int max_depth) {
    return 6 * (T + 1) > 12 * max_depth ? 6 * (T + 1) : 12 * max_depth;
}
__host__ __device__ static inline int lane_chain_slots(int n, int T, int max_depth, int n_refine) {
    return 3 * n + lane_wslots(T, max_depth) + 2 * T + (n_refine > 1 ? 2 * T : 0);
}

// CTA-per-chain kernel: shared-memory layout (byte offsets) -- topology {ref, meta, fragments, row offsets, records},
// the chain's coordinates X[3][n], per-atom (force, moment about t) AF[6][n] and a reduction scratch
struct CtaLayout { size_t ref, meta, frag, rows, recs, tt, masks, part, X, AF, PF, red, total; };
#define TRIDSK_AL16(x) (((x) + 15) / 16 * 16)
#define TRIDSK_CTA_WARPS 4             // the most warps a CTA kernel runs (score kernel, record instance: 128 threads)
__host__ __device__ static inline CtaLayout cta_layout(int n, int T, int n_pairs, bool dense) {
    CtaLayout L;
    size_t o = 0;
    const size_t npad = ((size_t)n + 31) / 32 * 32;
    L.ref = o; o += 16 * (size_t)n;
    L.meta = o; o = TRIDSK_AL16(o + 4 * (size_t)n);
    L.frag = o; o += sizeof(LaneFrag) * (size_t)(T + 1);
    L.rows = o; o = TRIDSK_AL16(o + 4 * (size_t)(n + 1));
    L.recs = o; o = TRIDSK_AL16(o + (dense ? 0 : 8 * 3 * (size_t)n_pairs));
    L.tt = o; o = TRIDSK_AL16(o + (dense ? 4 * 32 * 33 : 0));                     // float [32][33]: c of a pair of atom types
    L.masks = o; o = TRIDSK_AL16(o + (dense ? 4 * 4 * npad * (npad / 32) : 0));  // u32 [4][npad / 32][npad]: in the pair set, donor-acceptor; the same for l < b only
    L.part = o; o = TRIDSK_AL16(o + (dense ? 16 * npad * TRIDSK_CTA_WARPS : 0));   // per-warp partial forces, float4 [warps][npad]
    L.X = o; o = TRIDSK_AL16(o + (dense ? 16 * npad : 12 * (size_t)n));          // dense: float4 {x, y, z, 0} [npad], zero-padded
    L.AF = o; o = TRIDSK_AL16(o + 32 * (size_t)n);
    L.PF = o; o = TRIDSK_AL16(o + 32 * (size_t)n);
    L.red = o; o += 4 * 64;
    L.total = o;
    return L;
}
// threads per chain and lanes per atom of the CTA kernel (measured: 128 threads beat 256 also for 80-atom ligands, C4
// 122 vs 129 ms, because four CTAs per SM stay resident instead of two)
__host__ __device__ static inline void cta_shape(int n, int* threads, int* lpa) {
    if (n <= 16) { *threads = 128; *lpa = 8; }
    else if (n <= 32) { *threads = 128; *lpa = 4; }
    else if (n <= 64) { *threads = 128; *lpa = 2; }
    else { *threads = 128; *lpa = 1; }
}

// ---------------------------------------------------------------- host-side handles
struct tridsk_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    std::string err;
    long long launches = 0;
    int sm_count = 0;
    // scratch owned by the ctx (grown on demand)
    void* scratch[TRIDSK_SCRATCH] = {};
    size_t scratch_bytes[TRIDSK_SCRATCH] = {};
    void* pin = nullptr;          // pinned host staging block of tridsk_load_ligands (grown on demand)
    cudaEvent_t pin_ev = nullptr; // recorded after the last upload from the staging block
    size_t pin_bytes = 0;
    // cached CUDA graph of the last dock launch series
    cudaGraphExec_t graph_exec = nullptr;
    std::vector<unsigned char> graph_key;
    int graph_launches = 0;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};   // dock: before MC series, after MC series, after top-k
    bool ev_valid = false;
    cudaStream_t side[TRIDSK_BRANCHES] = {};           // side[0] unused
    cudaEvent_t fork_ev = nullptr, join_ev[TRIDSK_BRANCHES] = {};
    int kernel = 0;               // tridsk_set_kernel: 0 auto, 1 warp per chain, 2 lane per chain, 3 CTA per chain
    // grids come from a stream-ordered pool that keeps its memory (a screen rebuilds same-sized grids per receptor)
    cudaMemPool_t pool = nullptr;
    std::shared_ptr<bool> alive = std::make_shared<bool>(true);   // handles that outlive the ctx free synchronously
    int last_kernel = 0;          // what the last dock used
    // per-receptor grid cache (tridsk_build_grid_cached): most recently used first
    struct CacheEnt { unsigned long long key; size_t bytes; tridsk_grid* grid; };
    std::vector<CacheEnt> grid_cache;
    size_t cache_budget = (size_t)4 << 30, cache_bytes = 0;
    long long cache_hits = 0, cache_misses = 0;
};

struct tridsk_grid {
    tridsk_ctx* ctx;
    std::shared_ptr<bool> ctx_alive;
    int refs = 1;                 // handles out: the caller's, and the grid cache's if the grid is cached
    float* g = nullptr;
    float4* gp = nullptr;
    DGrid d;
    RecDev rd = {};               // tridsk_grid_attach_receptor: the receptor for the direct-pair mode
    void* rd_buf[4] = {nullptr, nullptr, nullptr, nullptr};   // atoms, cell_off, radius, role
};

struct tridsk_ligands {
    tridsk_ctx* ctx;
    int n_lig = 0, max_atoms = 0, max_tor = 0, min_atoms = 1 << 30;
    std::vector<LigHdr> hdr_h;
    std::vector<int> n_pairs;
    std::vector<int> bucket[TRIDSK_MAX_J + 1];   // ligand ids per J
    void* blob = nullptr;         // one device block holds all the packed arrays below
    LigHdr* hdr = nullptr;
    float4* atom_f4 = nullptr;
    int* atom_i = nullptr;
    FragRec* frags = nullptr;
    PairRound* rounds = nullptr;
    LaneFrag* lane_frags = nullptr;
    uint4* lane_stream = nullptr;
    LaneRec* lane_recs = nullptr;
    bool has_cta = false;
    int* cta_rows = nullptr;
    uint2* cta_recs = nullptr;
    float* cta_rtab = nullptr;
    // ligand ids by instance of the CTA kernel, [v][k]: k = 0 pair records, 1 dense partner sweep; v = which ligands are dense:
    // v = 0 those above TRIDSK_CTA_ROUNDS_N atoms (single docks: latency), v = 1 those above TRIDSK_CTA_DENSE_MIN (more chains
    // than the SMs hold at once: throughput)
    std::vector<int> cta_bucket[2][2];
    int* cta_bucket_dev[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};
    size_t cta_smem[2][2] = {{0, 0}, {0, 0}};    // largest shared-memory need per bucket
    int* all_ids = nullptr;       // 0..n_lig-1 re-ordered per lane bucket (refilled when the plan key changes)
    struct LaneBucket { int chains_per_cta; size_t smem; int first, count; int tm_cols; long long work = 0; int minb = 3; };   // tm_cols > 0: tensor-memory form, smem = bytes per warp
    std::vector<LaneBucket> lane_plan;
    std::vector<int> lane_ids_h;  // host copy behind all_ids (must outlive the async upload)
    long long lane_plan_key = -1; // n_chains << 8 | (n_refine > 1)
    int* bucket_dev[TRIDSK_MAX_J + 1] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    // the mixture-density term (tridsk_load_mdn); mdn.n_res == 0: absent
    MdnDev mdn = {};
    void* mdn_buf[9] = {};        // sph, res_off, rec, par, lig_off, cell_off, cell_at, dir_off, dir
};

// ---------------------------------------------------------------- kernel launchers (one per .cu)
cudaError_t launch_rec_pack(cudaStream_t s, const float* xyz, const int* type, int n_rec, int n_types, float4* out, int* bad);
cudaError_t launch_grid_build(cudaStream_t s, const float4* rec /* x,y,z,type */, int n_rec,
                              const float* pair_tab /* [n_types][n_types][4] */, int n_types,
                              const DParams& P, DGrid grid, float dc_max, const float* radius_h /* host [n_types] */,
                              const float* rec_radius_dev /* device [n_types] */, float* out);
cudaError_t launch_grid_pack(cudaStream_t s, DGrid grid, float4* out);
cudaError_t launch_mc(cudaStream_t s, int J, const McLaunch& a);
cudaError_t launch_mc_lane(cudaStream_t s, const McLaunch& a, int chains_per_cta, size_t smem_bytes, int minb);
cudaError_t launch_mc_lane_tm(cudaStream_t s, const McLaunch& a);
cudaError_t launch_score_lane(cudaStream_t s, const ScoreLaunch& a, int n_seg, size_t smem_bytes);
cudaError_t mc_lane_prepare(size_t max_smem_bytes);   // the *_prepare functions opt the kernels in to large shared memory on the CURRENT device
cudaError_t mc_cta_prepare();
cudaError_t topk_prepare();
cudaError_t launch_score(cudaStream_t s, const ScoreLaunch& a);
cudaError_t launch_mc_cta(cudaStream_t s, const McLaunch& a, int rounds /* 1: ligands above 64 atoms */, size_t smem_bytes);
cudaError_t launch_score_cta(cudaStream_t s, const ScoreLaunch& a, size_t smem_bytes);
cudaError_t launch_topk(cudaStream_t s, const TopkLaunch& a);
cudaError_t launch_score_direct(cudaStream_t s, const LigHdr* hdr, const float4* atom_f4, const int* atom_i, const LaneFrag* lane_frags,
                                const int* cta_rows, const uint2* cta_recs, const float4* rec, int n_rec, const float* radius,
                                const unsigned char* role, const DParams& P, const int* lig_index, const float* poses, int n_pose,
                                int pose_stride, float* energy, float* grad, int grad_stride, int max_atoms);
size_t topk_cluster_smem(int top_k, int max_atoms, int max_tor);
cudaError_t launch_mdn_spheres(cudaStream_t s, const float* res_xyz, const int* res_off, int n_res, float d_cut, float4* rec, float4* sph);
cudaError_t launch_mdn_cells(cudaStream_t s, const MdnDev& M, float cell, bool fill, int* counts_or_off, float4* cell_at);
cudaError_t launch_mdn_dir(cudaStream_t s, const MdnDev& M, bool fill, int* counts_or_off, int2* dir);
cudaError_t launch_mdn_pack(cudaStream_t s, const LigHdr* hdr, const int* atom_i, int n_lig, int n_res, int K, const long long* lig_off, const long long* in_off,
                            const float* pi, const float* mu, const float* sigma, float w_mdn, float4* par, int* bad);
cudaError_t launch_microbench(cudaStream_t s, int which, int sm_count, void* buf, size_t bytes, int iters, float* sink, double* work);
cudaError_t launch_philox_debug(cudaStream_t s, const unsigned int* ctr_key /* dev[6] */, unsigned int* out /* dev[4] */);
