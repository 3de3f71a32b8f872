// internal.h -- structures shared by the translation units of libtridsk (host + device).
// Nothing here is visible through the C-ABI (include/tridsk.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/tridsk.h"

#define TRIDSK_WARPS_PER_CTA 4
#define TRIDSK_MAX_J 4           // atoms per lane (n_atoms <= 32 * MAX_J)
#define TRIDSK_MAX_TILES 10      // J(J+1)/2 tiles of the pair schedule

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
    int nx, ny, nz, n_types;
    size_t plane;                 // nx*ny*nz
    float ox, oy, oz, h, inv_h;
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
    int pad[4];
};

// Per-fragment record; fragment 0 is the root, fragment k+1 hangs off torsion k.
struct FragRec {
    float ux, uy, uz, ox;         // axis unit vector and axis point (atom b_k), reference frame
    float oy, oz, pad0, pad1;
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
    const int* lig_list;          // ligands handled by this launch (one J bucket)
    int n_list;
    DGrid grid;
    DParams P;
    float box_min[3], box_max[3], centre[3], radius;
    int n_chains, pose_stride;
    int chain_base;               // global id of local chain 0 in the Philox counter (multi-GPU chain sharding)
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
};

struct ScoreLaunch {
    const LigHdr* hdr;
    const float4* atom_f4;
    const int* atom_i;
    const FragRec* frags;
    const PairRound* rounds;
    DGrid grid;
    DParams P;
    const int* lig_index;
    const float* poses;
    int n_pose, pose_stride;
    float* energy;                // [n_pose][3]
    float* grad; int grad_stride;
    float* coords; int coord_stride;
};

struct TopkLaunch {
    const LigHdr* hdr;
    const float* e_best; const float* pose_best;
    int n_lig, n_chains, pose_stride, top_k;
    float w_tor;
    float* out_energy; float* out_pose; int* out_chain;
};

// ---------------------------------------------------------------- host-side handles
struct tridsk_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    std::string err;
    long long launches = 0;
    int sm_count = 0;
    // scratch owned by the ctx (grown on demand)
    void* scratch[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    size_t scratch_bytes[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    // cached CUDA graph of the last dock launch series
    cudaGraphExec_t graph_exec = nullptr;
    std::vector<unsigned char> graph_key;
    int graph_launches = 0;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};   // dock: before MC series, after MC series, after top-k
    bool ev_valid = false;
};

struct tridsk_grid {
    tridsk_ctx* ctx;
    float* g = nullptr;
    DGrid d;
};

struct tridsk_ligands {
    tridsk_ctx* ctx;
    int n_lig = 0, max_atoms = 0, max_tor = 0;
    std::vector<LigHdr> hdr_h;
    std::vector<int> n_pairs;
    std::vector<int> bucket[TRIDSK_MAX_J + 1];   // ligand ids per J
    LigHdr* hdr = nullptr;
    float4* atom_f4 = nullptr;
    int* atom_i = nullptr;
    FragRec* frags = nullptr;
    PairRound* rounds = nullptr;
    int* bucket_dev[TRIDSK_MAX_J + 1] = {nullptr, nullptr, nullptr, nullptr, nullptr};
};

// ---------------------------------------------------------------- kernel launchers (one per .cu)
cudaError_t launch_grid_build(cudaStream_t s, const float4* rec /* x,y,z,type */, int n_rec,
                              const float* pair_tab /* [n_types][n_types][4] */, int n_types,
                              const DParams& P, DGrid grid, float dc_max, float* out);
cudaError_t launch_mc(cudaStream_t s, int J, const McLaunch& a);
cudaError_t launch_score(cudaStream_t s, const ScoreLaunch& a);
cudaError_t launch_topk(cudaStream_t s, const TopkLaunch& a);
cudaError_t launch_philox_debug(cudaStream_t s, const unsigned int* ctr_key /* dev[6] */, unsigned int* out /* dev[4] */);
