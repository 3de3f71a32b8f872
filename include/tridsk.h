/*
 * tridsk.h -- C-ABI of libtridsk: batched gradient-guided Monte Carlo conformation sampling
 * (the hot path of TRIDS, arxiv 2510.24186) as hand-written CUDA for sm_100a, one GPU.
 *
 * Citations: P:N = /root/reference/PAPER.md line N.  O1..O13 / G1..G19 = DESIGN.md section 3
 * (the readings taken where the paper is silent or garbled).  The problem the four main calls
 * solve is the paper's statement of docking: given a receptor pocket, one or many
 * ligands with rotatable bonds and a search box, sample pose degrees of freedom (translation,
 * rotation, torsions) by Metropolis Monte Carlo with gradient refinement (P:143-148,
 * Fig. 2) under the score E_dock, and return the top-N lowest-score poses.
 *
 * Conventions
 *   - Every function returns TRIDSK_OK (0) or a negative error code and never aborts;
 *     tridsk_last_error(ctx) gives the text (valid until the next call on that ctx).
 *   - Pointers marked [host] must be host memory; [host|dev] may be either and are detected with
 *     cudaPointerGetAttributes.  The caller owns every input buffer (copied or consumed before the
 *     call returns) and every output buffer; the library owns what the opaque handles point to
 *     until the matching free.
 *   - All GPU work is enqueued on the stream given to tridsk_create.  Calls that write HOST
 *     outputs synchronise that stream before returning; calls that write only DEVICE outputs do not.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with TRIDSK_ECUDA.
 *   - Pose layout   [tx,ty,tz, qw,qx,qy,qz, theta_0..theta_{T-1}]  (Hamilton, active rotation,
 *     torsion k right-handed about tor_a[k] -> tor_b[k]; theta = 0, q = 1, t = 0 is ref_xyz; O8/G10).
 *     Input quaternions are renormalised; a pose whose quaternion has zero or non-finite norm is rejected with
 *     TRIDSK_EINVAL when the poses are HOST memory (tridsk_score_grad, tridsk_score_direct, tridsk_dock init_poses).
 *     Poses handed over in DEVICE memory are never read by the host (the call stays asynchronous): there such a pose
 *     gets NaN energies (tridsk_score_grad) or a chain that rejects every proposal (tridsk_dock).
 *   - Gradient layout [dE/dt (3), dE/domega (3, world-frame rotation vector about t), dE/dtheta (T)] (O9).
 *   - Limits: n_atoms <= 128, n_torsions <= 31, n_types <= 32 per ligand (TRIDSK_ELIMIT otherwise).
 */
#ifndef TRIDSK_H
#define TRIDSK_H

#ifdef __cplusplus
extern "C" {
#endif

#define TRIDSK_OK      0
#define TRIDSK_EINVAL (-1)   /* bad argument or inconsistent ligand topology */
#define TRIDSK_ENOMEM (-2)
#define TRIDSK_ECUDA  (-3)   /* CUDA error; text in tridsk_last_error */
#define TRIDSK_ELIMIT (-4)   /* a size limit above is exceeded */

#define TRIDSK_MAX_ATOMS    128
#define TRIDSK_MAX_TORSIONS 31
#define TRIDSK_MAX_TYPES    32

typedef struct tridsk_ctx tridsk_ctx;         /* owns CUDA resources on one device */
typedef struct tridsk_grid tridsk_grid;       /* owns the fp32 [n_types][nz][ny][nx] device grid */
typedef struct tridsk_ligands tridsk_ligands; /* owns the packed ligand batch on the device */

/* Every constant of the method; tridsk_default_params fills the paper's values. */
typedef struct {
    float w_long, w_clash, w_hbond;             /* 0.2, 10.0, 0.6    Eq.E_dock weights            */
    float long_mu, long_two_sigma2, long_dmax;  /* 3.0, 4.0, 10.0    Eq.E_long; G2            */
    float hb_mu, hb_sigma, hb_dmax, hb_dclash;  /* 2.88, 0.3, 3.4, 2.6   Eq.E_Hbond, Eq.E_clash */
    float d_floor, k_wall;                      /* 0.05 A, 10.0 /A^2  G4, G8                             */
    float beta, lr, adam_b1, adam_b2, adam_eps; /* 0.069, 0.1, 0.9, 0.999, 1e-8   P:148, G12      */
    float pert_trans, pert_rot;                 /* 2.0 A, 0.5 rad     G11                                 */
    float w_tor;                                /* 0.01               Eq.E_screen                  */
    int   n_refine;                             /* 1                  Adam steps per MC step, G12         */
} tridsk_params;

/* Atom-type table (O1): per type a vdW radius [A] and an H-bond role (bit0 donor, bit1 acceptor). [host] */
typedef struct {
    int n_types;
    const float* radius;
    const unsigned char* hb_role;
} tridsk_types;

/*
 * CSR-packed ligand batch, all [host], copied during tridsk_load_ligands.
 *   atom_off[n_lig+1]; ref_xyz[sum n][3] reference conformer (centred on its centroid, G10);
 *   atom_type[sum n]; atom_frag[sum n]: 0 = root rigid fragment, k+1 = the fragment hanging off
 *   torsion k (it moves with torsion k and all of k's ancestors);
 *   tor_off[n_lig+1]; tor_a/tor_b[sum T]: rotation axis a -> b, a on the root side;
 *   tor_parent[sum T]: parent torsion or -1; parents precede children.
 *   Intra-ligand pairs (O6): give them as pair_off[n_lig+1] + pair_ab[sum P][2], or pass
 *   pair_off = NULL and give the bond graph (bond_off[n_lig+1], bond_ab[sum nb][2]); the library
 *   then derives pairs = {a<b : bond-graph distance >= 4 and atom_frag[a] != atom_frag[b]}.
 *   Atom / torsion indices inside a ligand are local (0-based) bytes.
 */
typedef struct {
    int n_lig;
    const int* atom_off;
    const float* ref_xyz;
    const unsigned char* atom_type;
    const unsigned char* atom_frag;
    const int* tor_off;
    const unsigned char* tor_a;
    const unsigned char* tor_b;
    const signed char* tor_parent;
    const int* pair_off;
    const unsigned char* pair_ab;
    const int* bond_off;
    const unsigned char* bond_ab;
} tridsk_ligand_batch;

/* One record of the optional per-step trace of tridsk_dock (parity tests). */
typedef struct {
    float e_prop;   /* energy of the refined proposal (E_new, O12)          */
    float e_cur;    /* energy of the current accepted state before the step */
    float u;        /* the Metropolis uniform                               */
    int   flags;    /* bit0 = accepted; bits 8.. = perturbed entity (0 translation, 1 rotation, 2+k torsion k) */
} tridsk_trace_rec;

/* Optional controls of tridsk_dock; NULL = all zero = defaults. */
typedef struct {
    int first_step;            /* Philox step counter of the first MC step of this call (resume)            */
    const float* init_poses;   /* [host|dev] NULL -> Philox initialisation (O11); else [n_lig][n_chains][pose_stride] */
    int resume;                /* 1: start from chain_state (as written by an earlier call) instead of initialising   */
    float* chain_state;        /* [host|dev] NULL, or n_lig*n_chains*(2*pose_stride+2) floats laid out as four arrays
                                  {pose_cur[n_lig][n_chains][pose_stride], pose_best[same], E_cur[n_lig][n_chains],
                                  E_best[same]}; read if resume, always written                                       */
    tridsk_trace_rec* trace;   /* [host|dev] NULL, or [n_lig][n_chains][n_steps]                                      */
    int steps_per_launch;      /* MC steps per kernel launch; 0 = all n_steps in one launch                           */
    int no_graph;              /* 1: plain stream launches instead of a captured CUDA graph                           */
    int chain_base;            /* Philox chain id of local chain 0 (chain sharding across GPUs; results then do not
                                  depend on the GPU count)                                                            */
    float cluster_rmsd;        /* > 0: duplicate removal in the top-k ("clustered to remove the duplicates"; G20):
                                  chains are walked in (E_best, chain id) order and a pose whose heavy-atom RMSD (same
                                  atom order, receptor frame) to an already kept pose is below this many Angstrom is
                                  skipped.  Slots left over get chain -1, energies +inf and a zero pose.  Needs
                                  top_k * max_atoms <= 4096.  0: plain top-k (O13)                                     */
    int receptor_direct;       /* 1: the receptor term of every evaluation is the paper's own direct sum over the receptor atoms
                                  within the pair function's range (P:103-125, P:353 item 4) instead of the
                                  trilinear grid lookup: no interpolation error, no wall, ~500 pair evaluations per ligand atom.
                                  Needs tridsk_grid_attach_receptor on the grid; runs under the CTA-per-chain mapping (single
                                  docks, without E_MDN) and the warp-per-chain mapping (everything else)                     */
    int lig_base;              /* Philox ligand id of the handle's ligand 0: a batch docked in parts (tridsk_screen) draws the
                                  same random streams as the whole batch in one call                                         */
} tridsk_dock_opts;

/* ---- lifetime ------------------------------------------------------------------------------ */
/* cuda_stream: a cudaStream_t (e.g. torch.cuda.Stream().cuda_stream); NULL -> the ctx creates and owns a
 * non-blocking stream (the legacy default stream cannot be captured into a CUDA graph). */
int  tridsk_create(tridsk_ctx** out, int device, void* cuda_stream);
void tridsk_destroy(tridsk_ctx* ctx);
const char* tridsk_last_error(const tridsk_ctx* ctx);
void tridsk_default_params(tridsk_params* p);
int  tridsk_synchronize(tridsk_ctx* ctx);

/* ---- receptor grid (hot-path step a0; O3/O4) ------------------------------------------------- */
/*
 * G[t][k][j][i] = sum over receptor atoms a of e(s_a, t, |origin + spacing*(i,j,k) - r_a|), x fastest,
 * where e = w_long*L + w_clash*C + w_Hbond*H are the paper's receptor-ligand pair terms
 * (Eq.E_long, Eq.E_clash, Eq.E_Hbond; they depend on the ligand atom only through
 * its type, which is what makes the tabulation valid -- G7).  rec_xyz[n_rec][3], rec_type[n_rec]: [host|dev].
 * origin[3], dims[3] = (nx,ny,nz): [host].
 */
int tridsk_build_grid(tridsk_ctx* ctx, const float* rec_xyz, const int* rec_type, int n_rec,
                      const tridsk_types* types, const tridsk_params* params,
                      const float origin[3], const int dims[3], float spacing, tridsk_grid** out);
/*
 * The same grid through the ctx's per-receptor cache (many-target screens rebuild the same receptors'
 * grids over and over -- DEKOIS 2.0 has 81 targets; crystallographic waters kept as fixed receptor atoms, are
 * simply more rec_xyz rows and make a different key).  The key is a 64-bit hash of everything the grid depends on
 * (receptor coordinates and types, the type table, the pair-function parameters, origin / dims / spacing); a hit returns
 * the cached grid without launching anything, a miss builds it and keeps it.  The cache holds its own reference: free the
 * returned handle with tridsk_free_grid as usual.  Least recently used grids are dropped when the byte budget
 * (tridsk_grid_cache_config; default 4 GiB, 0 disables caching) is exceeded.  Receptor arrays in DEVICE memory are copied
 * to the host to be hashed.
 */
int tridsk_build_grid_cached(tridsk_ctx* ctx, const float* rec_xyz, const int* rec_type, int n_rec,
                             const tridsk_types* types, const tridsk_params* params,
                             const float origin[3], const int dims[3], float spacing, tridsk_grid** out);
/* budget_bytes >= 0 sets the budget (dropping grids beyond it); stats (may be NULL) [host] <- {hits, misses, grids held, bytes held}. */
int tridsk_grid_cache_config(tridsk_ctx* ctx, long long budget_bytes, long long stats[4]);

/* Give a grid the receptor it tabulates, for tridsk_dock's receptor_direct mode: the atoms are sorted into cells of a third of
 * the pair function's range (max of long_dmax, hb_dmax and the largest clash distance).  rec_xyz, rec_type: [host|dev]. */
int tridsk_grid_attach_receptor(tridsk_ctx* ctx, tridsk_grid* grid, const float* rec_xyz, const int* rec_type, int n_rec,
                                const tridsk_types* types, const tridsk_params* params);

/* Adopt a caller-built grid (e.g. the oracle's), copied from `values` [host|dev] [n_types][nz][ny][nx]. */
int tridsk_grid_from_values(tridsk_ctx* ctx, const float* values, int n_types,
                            const float origin[3], const int dims[3], float spacing, tridsk_grid** out);
/* Copy the grid out, dst [host|dev] [n_types][nz][ny][nx]. */
int tridsk_grid_export(tridsk_ctx* ctx, const tridsk_grid* grid, float* dst);
void tridsk_free_grid(tridsk_grid* grid);

/* ---- ligands ---------------------------------------------------------------------------------- */
int tridsk_load_ligands(tridsk_ctx* ctx, const tridsk_ligand_batch* batch, const tridsk_types* types,
                        tridsk_ligands** out);
/* n_pairs_out[n_lig] [host] (may be NULL): number of intra-ligand pairs per ligand (given or derived). */
int tridsk_ligand_info(const tridsk_ligands* ligs, int* n_lig, int* max_atoms, int* max_torsions, int* n_pairs_out);
void tridsk_free_ligands(tridsk_ligands* ligs);

/* ---- the mixture-density term E_MDN (O15) ---------------------------------- */
/*
 * The paper's main scoring term (w_MDN = 1.0):  E_MDN = - sum_i sum_j [d_ij < d_cut] sum_k pi_ijk N(d_ij; mu_ijk,
 * sigma_ijk)  (Eq.E_MDN; Eq.GMM) over pocket residues i and ligand atoms j, d_ij = the minimum distance
 * between the atoms of residue i and ligand atom j, d_cut = 5 A, N the normalised Gaussian density (G17).
 * The mixture parameters are the output of the paper's graph transformer, which is NOT part of this library:
 * the caller supplies them (bench.py and the tests: synthetic ones).
 *   n_res, res_off[n_res+1], res_xyz[res_off[n_res]][3]: the residues' atoms, [host];
 *   K; pi, mu, sigma: [host|dev], ligand-major: for ligand l of the batch a block [n_res][n_atoms(l)][K], atoms in the
 *   caller's order, blocks in batch order; sigma > 0.
 */
typedef struct {
    int n_res;
    const int* res_off;
    const float* res_xyz;
    int K;
    const float* pi;
    const float* mu;
    const float* sigma;
    float w_mdn;               /* 1.0 */
    float d_cut;               /* 5.0 */
} tridsk_mdn;
/* Attach the term to a ligand batch (NULL detaches it): every later tridsk_score_grad / tridsk_dock on these ligands
 * evaluates the full Eq.E_dock, E = w_MDN E_MDN + [grid terms] + E_intra; in tridsk_score_grad's energy[3]
 * the term is booked under "receptor" (it is a receptor-ligand term).  The gradient flows through the arg-min atom;
 * ties of the minimum go to the lowest atom index; the indicators are not differentiated (G21).  Parameters are copied. */
int tridsk_load_mdn(tridsk_ctx* ctx, tridsk_ligands* ligs, const tridsk_mdn* mdn);

/* ---- score + analytic gradient of given poses (steps a3..a6; O5..O9) --------------------------- */
/*
 * For pose i of ligand lig_index[i]: forward kinematics, E = sum_a [trilinear G_type(a)(x_a) + wall] + E_intra,
 * and the hand-derived gradient pushed back through the torsion tree (P:131, P:353 item 3).
 * lig_index[n_pose], poses[n_pose][pose_stride]: [host|dev], pose_stride >= 7 + max T.
 * energy[n_pose][3] = {total, receptor (inter), intra}; grad[n_pose][grad_stride] or NULL, grad_stride >= 6 + max T;
 * coords[n_pose][coord_stride][3] or NULL, coord_stride >= max n, atoms in the caller's order: [host|dev].
 */
int tridsk_score_grad(tridsk_ctx* ctx, const tridsk_grid* grid, const tridsk_ligands* ligs,
                      const tridsk_params* params, const int* lig_index, const float* poses, int n_pose,
                      int pose_stride, float* energy, float* grad, int grad_stride, float* coords, int coord_stride);

/*
 * The same evaluation with the receptor term taken the paper's own way (P:103-125, P:353 item 4):
 * direct sums over the receptor atoms, E_inter = sum_a sum_r e(s_r, t_a, |x_a - r_r|) -- no grid, no interpolation, no
 * wall.  It is what the grid tabulates (O3): the difference to tridsk_score_grad is the interpolation error of the hot
 * path's receptor term.  A measuring tool (O(n_atoms * n_rec) per pose), not part of tridsk_dock.
 * rec_xyz[n_rec][3], rec_type[n_rec], lig_index, poses, energy[n_pose][3], grad (or NULL): [host|dev] as in
 * tridsk_score_grad.  Needs a ligand batch of at most 1024 ligands.
 */
int tridsk_score_direct(tridsk_ctx* ctx, const float* rec_xyz, const int* rec_type, int n_rec, const tridsk_types* types,
                        const tridsk_params* params, const tridsk_ligands* ligs, const int* lig_index, const float* poses,
                        int n_pose, int pose_stride, float* energy, float* grad, int grad_stride);

/* ---- the docking run (steps a1..a10; O10..O13) ---------------------------------------------------- */
/*
 * For every ligand: n_chains independent chains x n_steps MC steps (perturb one entity -> n_refine
 * Adam steps on the analytic gradient -> Metropolis with a Philox4x32-10 stream keyed by
 * (seed; chain, step, ligand, purpose)), then the top_k lowest best-energies across chains
 * (ties -> lower chain id).
 * box_min/box_max/pocket_center: [host].  Outputs [host|dev]:
 *   out_energy[n_lig][top_k][2] = {E_dock, E_screen = E_dock/(1 + w_tor*T)};
 *   out_pose[n_lig][top_k][pose_stride]; out_chain[n_lig][top_k].  top_k <= n_chains.
 * opts->cluster_rmsd > 0 replaces the plain top-k by the duplicate-removing one (O14).
 */
int tridsk_dock(tridsk_ctx* ctx, const tridsk_grid* grid, const tridsk_ligands* ligs, const tridsk_params* params,
                const float box_min[3], const float box_max[3], const float pocket_center[3], float pocket_radius,
                int n_chains, int n_steps, int top_k, unsigned long long seed, int pose_stride,
                float* out_energy, float* out_pose, int* out_chain, const tridsk_dock_opts* opts);

/*
 * A whole screen in one call, from the caller's HOST ligand arrays: tridsk_load_ligands + tridsk_dock + tridsk_free_ligands,
 * but the batch goes in two parts and the host-side packing of the second (most of the batch) runs while the first is
 * docking on the GPU.  Results are identical to the three calls on the whole batch (the second part docks with
 * tridsk_dock_opts.lig_base = size of the first, so every chain draws the same Philox streams; "each of which was
 * individually tackled": ligands are independent).  Batches below 8,192 ligands go in one part.  Outputs [host|dev] as in
 * tridsk_dock, pose_stride >= 7 + the largest torsion count of the batch; the call returns when they are complete.  The
 * physics terms only: the mixture-density term is attached to a loaded batch (tridsk_load_mdn), which this call never exposes.
 */
int tridsk_screen(tridsk_ctx* ctx, const tridsk_grid* grid, const tridsk_ligand_batch* batch, const tridsk_types* types,
                  const tridsk_params* params, const float box_min[3], const float box_max[3],
                  const float pocket_center[3], float pocket_radius, int n_chains, int n_steps, int top_k,
                  unsigned long long seed, int pose_stride, float* out_energy, float* out_pose, int* out_chain);

/*
 * tridsk_dock for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the same docking run (a CTA per chain, Philox initialisation, plain top-k) whose only
 * scratch -- the per-chain state {pose_cur, pose_best, e_cur, e_best}, n_lig * n_chains * (2 * pose_stride + 2) floats --
 * lives in ONE array of TRIDSK_STATIC_SCRATCH_BYTES (4 MiB) that is part of the library image: every GPU that loads the
 * library holds it until the process exits.  The call makes no cudaMalloc / cudaFree / graph / event / stream creation;
 * it enqueues the fused MC kernel(s) and the top-k kernel on the ctx stream and returns without synchronising.
 *   - out_energy / out_pose / out_chain must be DEVICE memory (layout as tridsk_dock); TRIDSK_EINVAL otherwise.
 *   - TRIDSK_ELIMIT with a message naming both sizes when the chain state exceeds the 4 MiB (e.g. 1,024 chains of a
 *     20-torsion ligand need 0.22 MiB, 32 ligands x 384 chains x 6 torsions 1.3 MiB) or when the batch has more than
 *     1024 ligands (it needs the CTA-per-chain pair format); nothing is launched then.
 *   - The array is SHARED by every such call on that GPU, from any ctx or thread, and keeps the previous call's contents:
 *     two calls whose kernels overlap on the GPU (different streams, no ordering between them) race on it.  Calls on one
 *     stream are ordered and safe.  Nothing in it has to start at zero: the MC kernel writes every chain's state before
 *     the top-k kernel reads it.
 * Results are bit-identical to tridsk_dock under mapping 3 with the same arguments and no options.
 */
#define TRIDSK_STATIC_SCRATCH_BYTES (4u << 20)
int tridsk_dock_static(tridsk_ctx* ctx, const tridsk_grid* grid, const tridsk_ligands* ligs, const tridsk_params* params,
                       const float box_min[3], const float box_max[3], const float pocket_center[3], float pocket_radius,
                       int n_chains, int n_steps, int top_k, unsigned long long seed, int pose_stride,
                       float* out_energy, float* out_pose, int* out_chain);

/*
 * Chain-to-thread mapping of the fused kernel: 0 = automatic (measured crossovers: a CTA per chain for a single
 * dock -- up to 3 chains per SM, 5 when no ligand has 32 atoms or fewer --, a lane per chain from 64 chains per SM, a warp per
 * chain in between; batches of ligands above 64 atoms only: a CTA per chain up to 76 chains per SM, a lane per chain beyond; with
 * the mixture-density term attached: a CTA per chain up to 330 chains per SM, a lane per chain beyond), 1 = always
 * a warp per chain, 2 = always a lane per chain, 3 = always a CTA per chain (batches of at most 1024 ligands),
 * 4 = a lane per chain with the chains' coordinates in tensor memory (tcgen05.st/ld) for ligands of at most 42 atoms
 * where that keeps more warps resident -- same arithmetic and results as 2; experimental, never chosen automatically.
 * Applies to tridsk_dock and tridsk_score_grad on this ctx.  All mappings compute O1..O13; their fp32 summation orders
 * differ, so chains are bit-reproducible per mapping, not across mappings.
 */
int tridsk_set_kernel(tridsk_ctx* ctx, int kernel);
/* The mapping (1, 2 or 3) the last tridsk_dock on this ctx used; 0 before any dock. */
int tridsk_last_kernel(const tridsk_ctx* ctx);

/* Device time of the last tridsk_dock on this ctx, from CUDA events recorded on the ctx stream around the fused MC
 * kernel series and the top-k kernel: ms[0] = MC series, ms[1] = top-k.  Blocks until that dock has finished. [host] */
int tridsk_last_dock_ms(tridsk_ctx* ctx, float ms[2]);

/* Kernel launches enqueued by this ctx since creation (bench.py's gpu_launches). */
long long tridsk_launch_count(const tridsk_ctx* ctx);

/* Philox4x32-10 block for the given counter/key, computed ON THE DEVICE by the same routine the chains use
 * (test hook for O10).  ctr[4], key[2], out[4]: [host]. */
int tridsk_debug_philox(tridsk_ctx* ctx, const unsigned int ctr[4], const unsigned int key[2], unsigned int out[4]);

/*
 * The roofline denominators of the fused MC step, measured on this device: one launch of
 * microbenchmark `which` on the ctx stream, timed with CUDA events.  ms [host]: device time of the launch; work [host]:
 * what it did -- flops (TRIDSK_MB_FFMA, TRIDSK_MB_FFMA2: independent FP32 FMA chains, plain and packed f32x2), MUFU
 * operations (TRIDSK_MB_MUFU: ex2.approx chains), bytes read (TRIDSK_MB_L2_READ: coalesced 16-byte loads over a buffer of
 * `bytes`, `iters` passes; below the L2 size the buffer is L2-resident after the first pass), bytes of 32-byte sectors
 * touched (TRIDSK_MB_GATHER: per lane one 16-byte load from a pseudo-random sector of a buffer of `bytes`, the access a
 * trilinear lookup in the cell-packed grid makes once per atom).  Not on the docking path.
 */
#define TRIDSK_MB_FFMA    0
#define TRIDSK_MB_FFMA2   1
#define TRIDSK_MB_MUFU    2
#define TRIDSK_MB_L2_READ 3
#define TRIDSK_MB_GATHER  4
int tridsk_debug_microbench(tridsk_ctx* ctx, int which, unsigned long long bytes, int iters, float* ms, double* work);

#ifdef __cplusplus
}
#endif
#endif /* TRIDSK_H */
