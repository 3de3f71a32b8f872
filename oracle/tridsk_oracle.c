/*
 * oracle/tridsk_oracle.c -- plain fp64 CPU oracle for the TRIDS sampling hot path.
 *
 * TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code with the CUDA path
 * (paper_2510_24186_b200/csrc) and neither imports the other.
 *
 * Everything here is scalar, one chain at a time, in the paper's order and notation, with no
 * blocking, fusion or reordering; OpenMP is used ONLY over independent chains / grid nodes.
 * P:N = /root/reference/PAPER.md line N.  O1..O13 / G1..G19 = DESIGN.md section 3 (the readings
 * taken where the paper is silent, ambiguous or garbled).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): two-atom closed forms and the paper's printed
 * constants for the pair function; brute force == grid at nodes; trilinear exact on nodes and on
 * trilinear fields + scipy RegularGridInterpolator; FK vs scipy Rotation / textbook matrices /
 * preserved internal coordinates; intra-ligand rigid invariance + Newton's third law; analytic
 * gradient vs central differences; Philox known answers; Adam vs torch.optim.Adam; Metropolis
 * P(accept | dE = 10) = 0.5016; E_MDN (orc_mdn_energy): closed forms, scipy.stats.norm, central differences,
 * the plain Python transcription of the same definition (oracle/mdn.py), and total = physics + w_MDN E_MDN on a hand case.
 * PARITY UNPINNED: the whole stochastic chain (orc_dock) has no external truth -- the paper
 * prints no worked example -- so it is pinned only through its parts plus sanity invariants.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    double w_long, w_clash, w_hbond;             /* 0.2, 10.0, 0.6 */
    double long_mu, long_two_sigma2, long_dmax;  /* 3.0, 4.0, 10.0              P:113, G2 */
    double hb_mu, hb_sigma, hb_dmax, hb_dclash;  /* 2.88, 0.3, 3.4, 2.6 */
    double d_floor, k_wall;                      /* 0.05, 10.0                  G4, G8 */
    double beta, lr, adam_b1, adam_b2, adam_eps; /* 0.069, 0.1, .9, .999, 1e-8  P:148, G12 */
    double pert_trans, pert_rot;                 /* 2.0, 0.5                    G11 */
    double w_tor;                                /* 0.01 */
    int n_refine;                                /* 1                           G12 */
    int clash_literal;                           /* 0; 1 = paper-literal [d < d_vdw] indicator (G3) */
} orc_params;

typedef struct {
    int n_types;
    const double* radius;        /* [n_types] vdW radius, A */
    const unsigned char* role;   /* [n_types] bit0 donor, bit1 acceptor */
} orc_types;

typedef struct {
    const float* g;              /* fp32 [n_types][nz][ny][nx], x fastest (O4) */
    int n_types, nx, ny, nz;
    double origin[3], spacing;
    /* direct-pair receptor mode (the paper's own evaluation, P:103-125, P:353 item 4): when n_rec >= 0 and
     * rec_xyz != NULL the receptor term of orc_score_grad (hence of orc_mc_step / orc_dock) is the plain sum over these receptor
     * atoms -- no grid, no interpolation, no wall -- exactly as in orc_score_grad_direct */
    const double* rec_xyz;
    const int* rec_type;
    int n_rec;
} orc_grid;

/* O15: the mixture-density term of one (receptor, ligand) pair -- Eq.GMM, Eq.E_MDN */
typedef struct {
    int n_res, K;
    const int* res_off;          /* [n_res+1]: the atoms of residue i are res_xyz[res_off[i] .. res_off[i+1]) */
    const double* res_xyz;       /* [res_off[n_res]][3] */
    const double* pi;            /* [n_res][n][K] mixture weights of (residue i, ligand atom j) */
    const double* mu;            /* [n_res][n][K] */
    const double* sigma;         /* [n_res][n][K] */
    double w_mdn, d_cut;         /* 1.0, 5.0 A */
} orc_mdn;

typedef struct {
    int n, T, P;
    const double* ref;           /* [n][3] reference conformer, centred */
    const unsigned char* type;   /* [n] */
    const unsigned char* frag;   /* [n] 0 = root, k+1 = child fragment of torsion k */
    const unsigned char* tor_a;  /* [T] axis a -> b, a on the root side */
    const unsigned char* tor_b;
    const signed char* tor_parent; /* [T] -1 = root; parents precede children */
    const unsigned char* pairs;  /* [P][2] */
    const orc_mdn* mdn;          /* NULL: w_MDN E_MDN absent from the score (the round-1 hot path); else added to E */
} orc_ligand;

void orc_default_params(orc_params* p) {
    p->w_long = 0.2; p->w_clash = 10.0; p->w_hbond = 0.6;
    p->long_mu = 3.0; p->long_two_sigma2 = 4.0; p->long_dmax = 10.0;
    p->hb_mu = 2.88; p->hb_sigma = 0.3; p->hb_dmax = 3.4; p->hb_dclash = 2.6;
    p->d_floor = 0.05; p->k_wall = 10.0;
    p->beta = 0.069; p->lr = 0.1; p->adam_b1 = 0.9; p->adam_b2 = 0.999; p->adam_eps = 1e-8;
    p->pert_trans = 2.0; p->pert_rot = 0.5;
    p->w_tor = 0.01;
    p->n_refine = 1;
    p->clash_literal = 0;
}

/* ------------------------------------------------------------------ O2: pair function */
/* "acceptor/donor pair of hydrogen bond" */
static int hbpair(unsigned char rs, unsigned char rt) {
    return ((rs & 1) && (rt & 2)) || ((rs & 2) && (rt & 1));
}

/*
 * e(s,t,d) = w_long*L + w_clash*C + w_Hbond*H  (Eq.E_dock without the MDN term)
 *   L = -[d < d_max] exp(-(d - d_vdw - mu)^2 / (2 sigma^2))     Eq.E_long  P:111-113 (sign: G1)
 *   C = -[d < d_c]   ln(max(d, d_floor) / d_c)                   Eq.E_clash P:117-119 (G3, G4)
 *   H = -[hbpair and d < d_Hmax] exp(-(d - 2.88)^2 / (2*0.3^2))  Eq.E_Hbond
 * de/dd: derivative of the smooth part inside each indicator; jumps are not differentiated.
 */
void orc_pair(const orc_params* p, double rad_s, unsigned char role_s, double rad_t, unsigned char role_t,
              double d, double* e, double* dedd) {
    double dvdw = rad_s + rad_t;
    int hb = hbpair(role_s, role_t);
    double E = 0.0, D = 0.0;
    if (d < p->long_dmax) {
        double t = d - dvdw - p->long_mu;
        double g = exp(-t * t / p->long_two_sigma2);
        E += p->w_long * (-g);
        D += p->w_long * (2.0 * t / p->long_two_sigma2) * g;
    }
    double dc = hb ? p->hb_dclash : dvdw;
    double dind = p->clash_literal ? dvdw : dc;
    if (d < dind) {
        double dd = d > p->d_floor ? d : p->d_floor;
        E += p->w_clash * (-log(dd / dc));
        if (d > p->d_floor) D += p->w_clash * (-1.0 / d);
    }
    if (hb && d < p->hb_dmax) {
        double t = d - p->hb_mu;
        double s2 = p->hb_sigma * p->hb_sigma;
        double g = exp(-t * t / (2.0 * s2));
        E += p->w_hbond * (-g);
        D += p->w_hbond * (t / s2) * g;
    }
    *e = E; *dedd = D;
}

/* ------------------------------------------------- O3: receptor field, brute force (the paper's sums) */
/* F_t(x) = sum over receptor atoms a of e(s_a, t, |x - r_a|)  -- i over receptor, j = one ligand atom of type t */
double orc_field_brute(const orc_params* p, const orc_types* ty, const double* rec_xyz, const int* rec_type,
                       int n_rec, int t, const double x[3]) {
    double sum = 0.0;
    for (int a = 0; a < n_rec; ++a) {
        double dx = x[0] - rec_xyz[3 * a], dy = x[1] - rec_xyz[3 * a + 1], dz = x[2] - rec_xyz[3 * a + 2];
        double d = sqrt(dx * dx + dy * dy + dz * dz), e, de;
        int s = rec_type[a];
        orc_pair(p, ty->radius[s], ty->role[s], ty->radius[t], ty->role[t], d, &e, &de);
        sum += e;
    }
    return sum;
}

/* ------------------------------------------------- O4: grid = field sampled on nodes, rounded once to fp32 */
void orc_build_grid(const orc_params* p, const orc_types* ty, const double* rec_xyz, const int* rec_type, int n_rec,
                    const double origin[3], int nx, int ny, int nz, double spacing, float* out) {
    for (int t = 0; t < ty->n_types; ++t) {
#pragma omp parallel for collapse(2) schedule(static)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    double x[3] = {origin[0] + spacing * i, origin[1] + spacing * j, origin[2] + spacing * k};
                    out[(((size_t)t * nz + k) * ny + j) * nx + i] =
                        (float)orc_field_brute(p, ty, rec_xyz, rec_type, n_rec, t, x);
                }
    }
}

/* ------------------------------------------------- O5: trilinear interpolation + wall, value and gradient */
void orc_interp(const orc_params* p, const orc_grid* G, int t, const double x[3], double* e, double grad[3]) {
    int n[3] = {G->nx, G->ny, G->nz}, i0[3];
    double f[3], wall = 0.0, gw[3] = {0, 0, 0};
    int clamped[3];
    for (int c = 0; c < 3; ++c) {
        double u = (x[c] - G->origin[c]) / G->spacing;
        double uc = u < 0.0 ? 0.0 : (u > (double)(n[c] - 1) ? (double)(n[c] - 1) : u);
        clamped[c] = (uc != u);
        int i = (int)floor(uc);
        if (i > n[c] - 2) i = n[c] - 2;
        i0[c] = i;
        f[c] = uc - i;
        double xc = G->origin[c] + uc * G->spacing;         /* clamped position */
        double dx = clamped[c] ? x[c] - xc : 0.0;           /* wall acts only outside the grid */
        wall += p->k_wall * dx * dx;
        gw[c] = 2.0 * p->k_wall * dx;
    }
    const float* g = G->g + (size_t)t * G->nz * G->ny * G->nx;
    double v[2][2][2];
    for (int dz = 0; dz < 2; ++dz)
        for (int dy = 0; dy < 2; ++dy)
            for (int dx = 0; dx < 2; ++dx)
                v[dz][dy][dx] = (double)g[((size_t)(i0[2] + dz) * G->ny + (i0[1] + dy)) * G->nx + (i0[0] + dx)];
    double val = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
    for (int dz = 0; dz < 2; ++dz)
        for (int dy = 0; dy < 2; ++dy)
            for (int dx = 0; dx < 2; ++dx) {
                double wx = dx ? f[0] : 1.0 - f[0], wy = dy ? f[1] : 1.0 - f[1], wz = dz ? f[2] : 1.0 - f[2];
                double sx = dx ? 1.0 : -1.0, sy = dy ? 1.0 : -1.0, sz = dz ? 1.0 : -1.0;
                val += wx * wy * wz * v[dz][dy][dx];
                gx += sx * wy * wz * v[dz][dy][dx];
                gy += wx * sy * wz * v[dz][dy][dx];
                gz += wx * wy * sz * v[dz][dy][dx];
            }
    *e = val + wall;
    grad[0] = (clamped[0] ? 0.0 : gx / G->spacing) + gw[0];
    grad[1] = (clamped[1] ? 0.0 : gy / G->spacing) + gw[1];
    grad[2] = (clamped[2] ? 0.0 : gz / G->spacing) + gw[2];
}

/* ------------------------------------------------------------------ small vector / quaternion helpers */
static void quat_normalise(double q[4]) {
    double n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    q[0] /= n; q[1] /= n; q[2] /= n; q[3] /= n;
}
/* Hamilton product r = a (x) b, scalar first */
static void quat_mul(const double a[4], const double b[4], double r[4]) {
    r[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
    r[1] = a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2];
    r[2] = a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1];
    r[3] = a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0];
}
/* active rotation matrix of a unit quaternion */
static void quat_matrix(const double q[4], double R[3][3]) {
    double w = q[0], x = q[1], y = q[2], z = q[3];
    R[0][0] = 1 - 2 * (y * y + z * z); R[0][1] = 2 * (x * y - w * z);     R[0][2] = 2 * (x * z + w * y);
    R[1][0] = 2 * (x * y + w * z);     R[1][1] = 1 - 2 * (x * x + z * z); R[1][2] = 2 * (y * z - w * x);
    R[2][0] = 2 * (x * z - w * y);     R[2][1] = 2 * (y * z + w * x);     R[2][2] = 1 - 2 * (x * x + y * y);
}
/* exponential map: rotation vector v -> unit quaternion */
static void quat_exp(const double v[3], double q[4]) {
    double a = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    if (a < 1e-12) { q[0] = 1.0; q[1] = 0.5 * v[0]; q[2] = 0.5 * v[1]; q[3] = 0.5 * v[2]; quat_normalise(q); return; }
    double s = sin(0.5 * a) / a;
    q[0] = cos(0.5 * a); q[1] = s * v[0]; q[2] = s * v[1]; q[3] = s * v[2];
}

/* is torsion k equal to, or an ancestor of, the torsion that owns fragment f ? */
static int in_subtree(const orc_ligand* L, int f, int k) {
    int j = f - 1;                       /* fragment f is the child fragment of torsion f-1 */
    while (j >= 0) {
        if (j == k) return 1;
        j = L->tor_parent[j];
    }
    return 0;
}

/* ------------------------------------------------------------------ O8: forward kinematics */
/*
 * pose = [tx,ty,tz, qw,qx,qy,qz, theta_0..theta_{T-1}].  Start from the reference conformer; for
 * k = 0..T-1 (parents first) rotate every atom of subtree(k) about the CURRENT axis x[a_k] -> x[b_k]
 * by theta_k (Rodrigues, right-handed about a -> b); then x <- Rot(q) x + t  (P:141, P:353 item 3).
 */
void orc_fk(const orc_ligand* L, const double* pose, double* x /* [n][3] */) {
    memcpy(x, L->ref, sizeof(double) * 3 * L->n);
    for (int k = 0; k < L->T; ++k) {
        const double* a = x + 3 * L->tor_a[k];
        double b[3] = {x[3 * L->tor_b[k]], x[3 * L->tor_b[k] + 1], x[3 * L->tor_b[k] + 2]};
        double u[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]};
        double un = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        u[0] /= un; u[1] /= un; u[2] /= un;
        double c = cos(pose[7 + k]), s = sin(pose[7 + k]);
        for (int i = 0; i < L->n; ++i) {
            if (!in_subtree(L, L->frag[i], k)) continue;
            double v[3] = {x[3 * i] - b[0], x[3 * i + 1] - b[1], x[3 * i + 2] - b[2]};
            double ud = u[0] * v[0] + u[1] * v[1] + u[2] * v[2];
            double cr[3] = {u[1] * v[2] - u[2] * v[1], u[2] * v[0] - u[0] * v[2], u[0] * v[1] - u[1] * v[0]};
            for (int d = 0; d < 3; ++d)                      /* v c + (u x v) s + u (u.v)(1 - c) */
                x[3 * i + d] = b[d] + v[d] * c + cr[d] * s + u[d] * ud * (1.0 - c);
        }
    }
    double q[4] = {pose[3], pose[4], pose[5], pose[6]}, R[3][3];
    quat_normalise(q);
    quat_matrix(q, R);
    for (int i = 0; i < L->n; ++i) {
        double v[3] = {x[3 * i], x[3 * i + 1], x[3 * i + 2]};
        for (int d = 0; d < 3; ++d) x[3 * i + d] = R[d][0] * v[0] + R[d][1] * v[1] + R[d][2] * v[2] + pose[d];
    }
}

/* ------------------------------------------------------------------ O6: pair list from the bond graph */
/* pairs = { a < b : bond-graph distance >= 4 and frag[a] != frag[b] }  (G6, Vina-style 1-2/1-3/1-4 exclusion).
 * Returns P; writes at most cap pairs. */
int orc_derive_pairs(int n, const unsigned char* frag, const unsigned char* bonds, int n_bonds,
                     unsigned char* pairs, int cap) {
    int* dist = (int*)malloc(sizeof(int) * n * n);
    for (int i = 0; i < n * n; ++i) dist[i] = 1 << 20;
    for (int i = 0; i < n; ++i) dist[i * n + i] = 0;
    for (int b = 0; b < n_bonds; ++b) {
        int u = bonds[2 * b], v = bonds[2 * b + 1];
        dist[u * n + v] = dist[v * n + u] = 1;
    }
    for (int k = 0; k < n; ++k)                      /* Floyd-Warshall: plain definition of graph distance */
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j)
                if (dist[i * n + k] + dist[k * n + j] < dist[i * n + j]) dist[i * n + j] = dist[i * n + k] + dist[k * n + j];
    int P = 0;
    for (int a = 0; a < n; ++a)
        for (int b = a + 1; b < n; ++b)
            if (dist[a * n + b] >= 4 && frag[a] != frag[b]) {
                if (P < cap) { pairs[2 * P] = (unsigned char)a; pairs[2 * P + 1] = (unsigned char)b; }
                ++P;
            }
    free(dist);
    return P;
}

/* ------------------------------------------------------------------ O15: E_MDN */
/*
 * E_MDN = - sum_i sum_j [d_ij < d_cut] sum_k pi_ijk N(d_ij; mu_ijk, sigma_ijk)  (Eq.E_MDN, sign G1), with
 * N the normalised Gaussian density (G17) and d_ij the minimum distance between the atoms of residue i and ligand atom j
 * (P:93); ties of the minimum go to the lowest atom index, and neither the arg-min switch nor the cut-off indicator is
 * differentiated (G21): the gradient flows through the arg-min atom.
 * x [n][3] ligand coordinates.  *e = E_MDN (unweighted); g (may be NULL) [n][3] += nothing -- it is SET to dE_MDN/dx;
 * dmin (may be NULL) [n_res][n] the minimum distances.
 */
void orc_mdn_energy(const orc_mdn* M, int n, const double* x, double* e, double* g, double* dmin) {
    double E = 0.0;
    if (g) for (int c = 0; c < 3 * n; ++c) g[c] = 0.0;
    for (int i = 0; i < M->n_res; ++i) {
        for (int j = 0; j < n; ++j) {
            double best = INFINITY;
            int r_best = -1;
            for (int r = M->res_off[i]; r < M->res_off[i + 1]; ++r) {
                double dv[3] = {x[3 * j] - M->res_xyz[3 * r], x[3 * j + 1] - M->res_xyz[3 * r + 1], x[3 * j + 2] - M->res_xyz[3 * r + 2]};
                double d = sqrt(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]);
                if (d < best) { best = d; r_best = r; }
            }
            if (dmin) dmin[(size_t)i * n + j] = best;
            if (!(best < M->d_cut)) continue;
            double dE_dd = 0.0;
            for (int k = 0; k < M->K; ++k) {
                size_t q = ((size_t)i * n + j) * M->K + k;
                double sg = M->sigma[q], m = M->mu[q], w = M->pi[q];
                double N = exp(-(best - m) * (best - m) / (2.0 * sg * sg)) / (sg * sqrt(2.0 * M_PI));
                E -= w * N;
                dE_dd += w * N * (best - m) / (sg * sg);
            }
            if (g && best > 0.0)
                for (int c = 0; c < 3; ++c) g[3 * j + c] += dE_dd * (x[3 * j + c] - M->res_xyz[3 * r_best + c]) / best;
        }
    }
    *e = E;
}

/* ------------------------------------------------------------------ O7 + O9: score and gradient */
/* O9: pose gradient from the per-atom gradient g[n][3] by the direct sums (no tree accumulation), O(N*T). */
static void pose_gradient(const orc_ligand* L, const double* pose, const double* x, const double* g, double* grad) {
    int n = L->n;
    for (int c = 0; c < 6 + L->T; ++c) grad[c] = 0.0;
    for (int a = 0; a < n; ++a) {
        double r[3] = {x[3 * a] - pose[0], x[3 * a + 1] - pose[1], x[3 * a + 2] - pose[2]};
        const double* ga = g + 3 * a;
        grad[0] += ga[0]; grad[1] += ga[1]; grad[2] += ga[2];
        grad[3] += r[1] * ga[2] - r[2] * ga[1];
        grad[4] += r[2] * ga[0] - r[0] * ga[2];
        grad[5] += r[0] * ga[1] - r[1] * ga[0];
    }
    for (int k = 0; k < L->T; ++k) {
        const double* xa = x + 3 * L->tor_a[k];
        const double* xb = x + 3 * L->tor_b[k];
        double u[3] = {xb[0] - xa[0], xb[1] - xa[1], xb[2] - xa[2]};
        double un = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        u[0] /= un; u[1] /= un; u[2] /= un;
        double tq[3] = {0, 0, 0};
        for (int a = 0; a < n; ++a) {
            if (!in_subtree(L, L->frag[a], k)) continue;
            double r[3] = {x[3 * a] - xb[0], x[3 * a + 1] - xb[1], x[3 * a + 2] - xb[2]};
            const double* ga = g + 3 * a;
            tq[0] += r[1] * ga[2] - r[2] * ga[1];
            tq[1] += r[2] * ga[0] - r[0] * ga[2];
            tq[2] += r[0] * ga[1] - r[1] * ga[0];
        }
        grad[6 + k] = u[0] * tq[0] + u[1] * tq[1] + u[2] * tq[2];
    }
}

/*
 * E = sum_a [interp(a) + wall(a)] + E_intra (+ w_MDN E_MDN when L->mdn is set, O15; booked under inter).
 * energy[3] = {total, inter, intra}.
 * grad (may be NULL) = [dE/dt (3), dE/domega (3, world-frame rotation vector about t), dE/dtheta (T)]
 * by the direct sums of O9; coords (may be NULL) [n][3]; gatom (may be NULL) [n][3] = dE/dx_a.
 */
void orc_score_grad(const orc_params* p, const orc_types* ty, const orc_grid* G, const orc_ligand* L,
                    const double* pose, double energy[3], double* grad, double* coords, double* gatom) {
    int n = L->n;
    double* x = (double*)malloc(sizeof(double) * 3 * n);
    double* g = (double*)calloc(3 * n, sizeof(double));
    orc_fk(L, pose, x);
    double e_inter = 0.0, e_intra = 0.0;
    for (int a = 0; a < n; ++a) {
        if (G->rec_xyz) {                      /* direct sums over the receptor atoms (O3 evaluated at the atom itself) */
            int ta = L->type[a];
            for (int r = 0; r < G->n_rec; ++r) {
                double dv[3] = {x[3 * a] - G->rec_xyz[3 * r], x[3 * a + 1] - G->rec_xyz[3 * r + 1], x[3 * a + 2] - G->rec_xyz[3 * r + 2]};
                double d = sqrt(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]), e, de;
                int sr = G->rec_type[r];
                orc_pair(p, ty->radius[sr], ty->role[sr], ty->radius[ta], ty->role[ta], d, &e, &de);
                e_inter += e;
                if (d > 0.0)
                    for (int c = 0; c < 3; ++c) g[3 * a + c] += de * dv[c] / d;
            }
            continue;
        }
        double e, ga[3];
        orc_interp(p, G, L->type[a], x + 3 * a, &e, ga);
        e_inter += e;
        for (int d = 0; d < 3; ++d) g[3 * a + d] += ga[d];
    }
    for (int k = 0; k < L->P; ++k) {
        int a = L->pairs[2 * k], b = L->pairs[2 * k + 1];
        double dv[3] = {x[3 * a] - x[3 * b], x[3 * a + 1] - x[3 * b + 1], x[3 * a + 2] - x[3 * b + 2]};
        double d = sqrt(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]), e, de;
        int ta = L->type[a], tb = L->type[b];
        orc_pair(p, ty->radius[ta], ty->role[ta], ty->radius[tb], ty->role[tb], d, &e, &de);
        e_intra += e;
        if (d > 0.0)
            for (int c = 0; c < 3; ++c) {
                g[3 * a + c] += de * dv[c] / d;
                g[3 * b + c] -= de * dv[c] / d;
            }
    }
    if (L->mdn) {                              /* E_dock = w_MDN E_MDN + ...; a receptor-ligand term: booked under "inter" */
        double e_mdn, *gm = (double*)malloc(sizeof(double) * 3 * n);
        orc_mdn_energy(L->mdn, n, x, &e_mdn, gm, NULL);
        e_inter += L->mdn->w_mdn * e_mdn;
        for (int c = 0; c < 3 * n; ++c) g[c] += L->mdn->w_mdn * gm[c];
        free(gm);
    }
    energy[0] = e_inter + e_intra; energy[1] = e_inter; energy[2] = e_intra;
    if (grad) pose_gradient(L, pose, x, g, grad);
    if (coords) memcpy(coords, x, sizeof(double) * 3 * n);
    if (gatom) memcpy(gatom, g, sizeof(double) * 3 * n);
    free(x); free(g);
}

/*
 * The same pose evaluation with the receptor term taken the paper's own way (P:103-125, P:353 item 4): direct sums over
 * the receptor atoms, E_inter = sum_a sum_r e(s_r, t_a, |x_a - r_r|), no grid, no interpolation, no wall.
 * NEXT-3: it is what the grid tabulates (O3), so the difference to orc_score_grad is the interpolation error.
 */
void orc_score_grad_direct(const orc_params* p, const orc_types* ty, const double* rec_xyz, const int* rec_type, int n_rec,
                           const orc_ligand* L, const double* pose, double energy[3], double* grad, double* coords,
                           double* gatom) {
    int n = L->n;
    double* x = (double*)malloc(sizeof(double) * 3 * n);
    double* g = (double*)calloc(3 * n, sizeof(double));
    orc_fk(L, pose, x);
    double e_inter = 0.0, e_intra = 0.0;
    for (int a = 0; a < n; ++a) {
        int ta = L->type[a];
        for (int r = 0; r < n_rec; ++r) {
            double dv[3] = {x[3 * a] - rec_xyz[3 * r], x[3 * a + 1] - rec_xyz[3 * r + 1], x[3 * a + 2] - rec_xyz[3 * r + 2]};
            double d = sqrt(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]), e, de;
            int s = rec_type[r];
            orc_pair(p, ty->radius[s], ty->role[s], ty->radius[ta], ty->role[ta], d, &e, &de);
            e_inter += e;
            if (d > 0.0)
                for (int c = 0; c < 3; ++c) g[3 * a + c] += de * dv[c] / d;
        }
    }
    for (int k = 0; k < L->P; ++k) {
        int a = L->pairs[2 * k], b = L->pairs[2 * k + 1];
        double dv[3] = {x[3 * a] - x[3 * b], x[3 * a + 1] - x[3 * b + 1], x[3 * a + 2] - x[3 * b + 2]};
        double d = sqrt(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]), e, de;
        int ta = L->type[a], tb = L->type[b];
        orc_pair(p, ty->radius[ta], ty->role[ta], ty->radius[tb], ty->role[tb], d, &e, &de);
        e_intra += e;
        if (d > 0.0)
            for (int c = 0; c < 3; ++c) {
                g[3 * a + c] += de * dv[c] / d;
                g[3 * b + c] -= de * dv[c] / d;
            }
    }
    if (L->mdn) {                              /* E_dock = w_MDN E_MDN + ...; a receptor-ligand term: booked under "inter" */
        double e_mdn, *gm = (double*)malloc(sizeof(double) * 3 * n);
        orc_mdn_energy(L->mdn, n, x, &e_mdn, gm, NULL);
        e_inter += L->mdn->w_mdn * e_mdn;
        for (int c = 0; c < 3 * n; ++c) g[c] += L->mdn->w_mdn * gm[c];
        free(gm);
    }
    energy[0] = e_inter + e_intra; energy[1] = e_inter; energy[2] = e_intra;
    if (grad) pose_gradient(L, pose, x, g, grad);
    if (coords) memcpy(coords, x, sizeof(double) * 3 * n);
    if (gatom) memcpy(gatom, g, sizeof(double) * 3 * n);
    free(x); free(g);
}

/* ------------------------------------------------------------------ O10: Philox4x32-10 */
static void mulhilo(uint32_t a, uint32_t b, uint32_t* hi, uint32_t* lo) {
    uint64_t p = (uint64_t)a * (uint64_t)b;
    *hi = (uint32_t)(p >> 32); *lo = (uint32_t)p;
}
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0, lo0, hi1, lo1;
        mulhilo(0xD2511F53u, c0, &hi0, &lo0);
        mulhilo(0xCD9E8D57u, c2, &hi1, &lo1);
        uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
/* u = ((r >> 9) + 0.5) * 2^-23 : in (0,1), exact in fp32 and fp64 */
static double u01(uint32_t r) { return ((double)(r >> 9) + 0.5) * (1.0 / 8388608.0); }
/* counter = (chain, step, ligand, purpose), key = (seed lo, seed hi) */
void orc_uniform4(uint64_t seed, uint32_t chain, uint32_t step, uint32_t ligand, uint32_t purpose, double u[4]) {
    uint32_t ctr[4] = {chain, step, ligand, purpose}, key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, o[4];
    orc_philox4x32_10(ctr, key, o);
    for (int i = 0; i < 4; ++i) u[i] = u01(o[i]);
}

/* ------------------------------------------------------------------ O11: chain initialisation */
void orc_init_pose(const orc_ligand* L, uint64_t seed, uint32_t chain, uint32_t ligand,
                   const double centre[3], double radius, double* pose) {
    double u[4];
    orc_uniform4(seed, chain, 0, ligand, 2, u);          /* uniform in the pocket sphere */
    double rr = radius * cbrt(u[0]), z = 2.0 * u[1] - 1.0, phi = 2.0 * M_PI * u[2], s = sqrt(1.0 - z * z);
    pose[0] = centre[0] + rr * s * cos(phi);
    pose[1] = centre[1] + rr * s * sin(phi);
    pose[2] = centre[2] + rr * z;
    orc_uniform4(seed, chain, 0, ligand, 3, u);          /* Shoemake: uniform on S^3 */
    double s1 = sqrt(1.0 - u[0]), s2 = sqrt(u[0]), t1 = 2.0 * M_PI * u[1], t2 = 2.0 * M_PI * u[2];
    pose[3] = s2 * cos(t2); pose[4] = s1 * sin(t1); pose[5] = s1 * cos(t1); pose[6] = s2 * sin(t2);
    for (int k = 0; k < L->T; ++k) {                     /* torsions uniform in [-pi, pi), four per block */
        if (k % 4 == 0) orc_uniform4(seed, chain, 0, ligand, 4 + k / 4, u);
        pose[7 + k] = M_PI * (2.0 * u[k % 4] - 1.0);
    }
}

static double clampd(double v, double lo, double hi) { return v < lo ? lo : (v > hi ? hi : v); }
static double wrap_pi(double a) {                         /* into [-pi, pi) */
    a = fmod(a + M_PI, 2.0 * M_PI);
    if (a < 0) a += 2.0 * M_PI;
    return a - M_PI;
}

/* ------------------------------------------------------------------ O12: one MC step */
typedef struct {
    double e_prop, e_cur, u;   /* refined-proposal energy, current energy before the step, Metropolis uniform */
    int accept, entity;
    double min_abs_g;          /* smallest |g_i| fed to Adam in this step (parity tests skip sign-unstable steps) */
    double p_accept;           /* exp(-beta dE) */
} orc_step_rec;

/*
 * pose (in/out: current accepted state), e_cur (in/out).  P:143-148, Fig. 2:
 * perturb one entity -> n_refine Adam steps on the 6+T tangent components -> E_new -> Metropolis.
 */
void orc_mc_step(const orc_params* p, const orc_types* ty, const orc_grid* G, const orc_ligand* L,
                 uint64_t seed, uint32_t chain, uint32_t step, uint32_t ligand,
                 const double box_min[3], const double box_max[3],
                 double* pose, double* e_cur, orc_step_rec* rec) {
    int T = L->T, D = 6 + T;
    double* prop = (double*)malloc(sizeof(double) * (7 + T));
    double* g = (double*)malloc(sizeof(double) * D);
    double* m = (double*)calloc(D, sizeof(double));
    double* v = (double*)calloc(D, sizeof(double));
    memcpy(prop, pose, sizeof(double) * (7 + T));
    double u[4];
    orc_uniform4(seed, chain, step, ligand, 0, u);
    int entity = (int)floor(u[0] * (T + 2));
    if (entity > T + 1) entity = T + 1;
    if (entity == 0) {
        for (int c = 0; c < 3; ++c)
            prop[c] = clampd(prop[c] + p->pert_trans * (2.0 * u[1 + c] - 1.0), box_min[c], box_max[c]);
    } else if (entity == 1) {
        double w[3] = {p->pert_rot * (2.0 * u[1] - 1.0), p->pert_rot * (2.0 * u[2] - 1.0), p->pert_rot * (2.0 * u[3] - 1.0)};
        double dq[4], q[4] = {prop[3], prop[4], prop[5], prop[6]}, r[4];
        quat_exp(w, dq); quat_mul(dq, q, r); quat_normalise(r);
        memcpy(prop + 3, r, sizeof(r));
    } else {
        prop[7 + entity - 2] = M_PI * (2.0 * u[1] - 1.0);
    }
    double min_abs_g = 1e300;
    for (int r = 1; r <= p->n_refine; ++r) {
        double E[3];
        orc_score_grad(p, ty, G, L, prop, E, g, NULL, NULL);
        double delta[64 + 6];
        for (int c = 0; c < D; ++c) {
            if (fabs(g[c]) < min_abs_g) min_abs_g = fabs(g[c]);
            m[c] = p->adam_b1 * m[c] + (1.0 - p->adam_b1) * g[c];
            v[c] = p->adam_b2 * v[c] + (1.0 - p->adam_b2) * g[c] * g[c];
            double mh = m[c] / (1.0 - pow(p->adam_b1, r)), vh = v[c] / (1.0 - pow(p->adam_b2, r));
            delta[c] = -p->lr * mh / (sqrt(vh) + p->adam_eps);
        }
        for (int c = 0; c < 3; ++c) prop[c] = clampd(prop[c] + delta[c], box_min[c], box_max[c]);
        double dq[4], q[4] = {prop[3], prop[4], prop[5], prop[6]}, rq[4];
        quat_exp(delta + 3, dq); quat_mul(dq, q, rq); quat_normalise(rq);
        memcpy(prop + 3, rq, sizeof(rq));
        for (int k = 0; k < T; ++k) prop[7 + k] = wrap_pi(prop[7 + k] + delta[6 + k]);
    }
    double En[3];
    orc_score_grad(p, ty, G, L, prop, En, NULL, NULL, NULL);
    orc_uniform4(seed, chain, step, ligand, 1, u);
    double pa = exp(-p->beta * (En[0] - *e_cur));
    int accept = isfinite(En[0]) && (u[0] < pa);           /* G15: NaN/inf proposal is rejected */
    rec->e_prop = En[0]; rec->e_cur = *e_cur; rec->u = u[0]; rec->accept = accept; rec->entity = entity;
    rec->min_abs_g = min_abs_g; rec->p_accept = pa;
    if (accept) { memcpy(pose, prop, sizeof(double) * (7 + T)); *e_cur = En[0]; }
    free(prop); free(g); free(m); free(v);
}

/* ------------------------------------------------------------------ whole dock of one ligand (a1..a8) */
/*
 * init_poses: NULL -> O11, else [n_chains][pose_stride].  Outputs per chain: best energy, best pose,
 * final current energy / pose; trace (may be NULL) [n_chains][n_steps].  Top-k (O13) is a sort of
 * e_best by (energy, chain id), done by the caller.
 */
void orc_dock(const orc_params* p, const orc_types* ty, const orc_grid* G, const orc_ligand* L,
              uint64_t seed, uint32_t ligand, int n_chains, int first_step, int n_steps,
              const double box_min[3], const double box_max[3], const double centre[3], double radius,
              const double* init_poses, int pose_stride,
              double* e_best, double* pose_best, double* e_cur_out, double* pose_cur_out, orc_step_rec* trace) {
    int W = 7 + L->T;
#pragma omp parallel for schedule(dynamic, 1)
    for (int c = 0; c < n_chains; ++c) {
        double cur[7 + 64], best[7 + 64], E[3];
        if (init_poses) memcpy(cur, init_poses + (size_t)c * pose_stride, sizeof(double) * W);
        else orc_init_pose(L, seed, (uint32_t)c, ligand, centre, radius, cur);
        { double q[4] = {cur[3], cur[4], cur[5], cur[6]}; quat_normalise(q); memcpy(cur + 3, q, sizeof(q)); }
        orc_score_grad(p, ty, G, L, cur, E, NULL, NULL, NULL);
        double ec = E[0], eb = E[0];
        memcpy(best, cur, sizeof(double) * W);
        for (int s = 0; s < n_steps; ++s) {
            orc_step_rec rec;
            orc_mc_step(p, ty, G, L, seed, (uint32_t)c, (uint32_t)(first_step + s), ligand, box_min, box_max, cur, &ec, &rec);
            if (rec.accept && ec < eb) { eb = ec; memcpy(best, cur, sizeof(double) * W); }
            if (trace) trace[(size_t)c * n_steps + s] = rec;
        }
        e_best[c] = eb; e_cur_out[c] = ec;
        memcpy(pose_best + (size_t)c * pose_stride, best, sizeof(double) * W);
        memcpy(pose_cur_out + (size_t)c * pose_stride, cur, sizeof(double) * W);
    }
}

/* Batched pose evaluation (the parity surface of tridsk_score_grad), OpenMP over poses. */
void orc_score_grad_batch(const orc_params* p, const orc_types* ty, const orc_grid* G, const orc_ligand* L,
                          const double* poses, int n_pose, int pose_stride,
                          double* energy /* [n_pose][3] */, double* grad /* [n_pose][gstride] or NULL */, int gstride,
                          double* coords /* [n_pose][cstride][3] or NULL */, int cstride) {
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < n_pose; ++i)
        orc_score_grad(p, ty, G, L, poses + (size_t)i * pose_stride, energy + 3 * (size_t)i,
                       grad ? grad + (size_t)i * gstride : NULL,
                       coords ? coords + (size_t)i * cstride * 3 : NULL, NULL);
}

int orc_sizeof_params(void) { return (int)sizeof(orc_params); }
int orc_sizeof_step_rec(void) { return (int)sizeof(orc_step_rec); }
int orc_sizeof_ligand(void) { return (int)sizeof(orc_ligand); }
int orc_sizeof_mdn(void) { return (int)sizeof(orc_mdn); }
int orc_sizeof_grid(void) { return (int)sizeof(orc_grid); }
