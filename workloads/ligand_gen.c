/*
 * workloads/ligand_gen.c -- seeded synthetic ligand generator (test/bench harness).
 *
 * Holds NONE of the method's arithmetic (no scoring, no kinematics, no pair lists):
 * it only produces INPUTS -- a reference conformer, atom types, a bond tree, the
 * choice of rotatable bonds and the resulting rigid-fragment / torsion-tree labels --
 * that the fp64 oracle (oracle/) and the CUDA library (paper_2510_24186_b200/) both
 * consume.  Recipe: SURVEY.md section 8(d) "Ligand(n, T, n_types)", restated in
 * DESIGN.md section 4.
 *
 *   atom 0 at the origin, atom 1 at 1.5 A; every further atom bonds to a uniformly
 *   chosen atom of degree < 4 at 1.5 A in an exact tetrahedral direction relative to
 *   that atom's existing bonds (1 bond: random azimuth on the 109.47 deg cone; 2: one
 *   of the two remaining sp3 directions; 3: the last one); a placement is rejected if
 *   any non-bonded atom is closer than 2.2 A.  Rotatable bonds: T drawn uniformly
 *   without replacement from the bonds whose two ends both have degree >= 2.
 *   backbone > 0 (config C4): the first `backbone` atoms form a linear chain, the
 *   torsions sit on its interior bonds centred on the middle atom, which is the root.
 *
 * The RNG is splitmix64 keyed by (seed, ligand index): ligands are independent of one
 * another and of the thread count.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define MAXN 255
#define BOND 1.5
#define MIN_NB 2.2

typedef struct { uint64_t s; } rng_t;

static uint64_t rng_next(rng_t* r) {
    uint64_t z = (r->s += 0x9E3779B97F4A7C15ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static double rng_unif(rng_t* r) { return (double)(rng_next(r) >> 11) * (1.0 / 9007199254740992.0); }
static int rng_int(rng_t* r, int n) { return (int)(rng_unif(r) * n) % n; }

static void cross3(const double* a, const double* b, double* c) {
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}
static void unit3(double* a) {
    double n = sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
    a[0] /= n; a[1] /= n; a[2] /= n;
}

/* direction of a new sp3 bond at atom p given its existing unit bond directions */
static void new_direction(rng_t* r, int nb, double dirs[4][3], double* out) {
    const double cos_t = -1.0 / 3.0, sin_t = sqrt(8.0) / 3.0; /* 109.47 deg */
    if (nb == 0) {
        out[0] = 1; out[1] = 0; out[2] = 0;
    } else if (nb == 1) {
        const double* d = dirs[0];
        double h[3] = {1, 0, 0}, e1[3], e2[3];
        if (fabs(d[0]) > 0.9) { h[0] = 0; h[1] = 1; }
        cross3(d, h, e1); unit3(e1);
        cross3(d, e1, e2);
        double phi = 2.0 * M_PI * rng_unif(r);
        for (int c = 0; c < 3; ++c) out[c] = cos_t * d[c] + sin_t * (cos(phi) * e1[c] + sin(phi) * e2[c]);
    } else if (nb == 2) {
        double n[3];
        cross3(dirs[0], dirs[1], n); unit3(n);
        double sg = rng_unif(r) < 0.5 ? 1.0 : -1.0;
        for (int c = 0; c < 3; ++c) out[c] = -0.5 * (dirs[0][c] + dirs[1][c]) + sg * sqrt(2.0 / 3.0) * n[c];
        unit3(out);
    } else {
        for (int c = 0; c < 3; ++c) out[c] = -(dirs[0][c] + dirs[1][c] + dirs[2][c]);
        unit3(out);
    }
}

/*
 * Returns 0 on success, <0 if the ligand could not be grown.
 *   xyz[n][3] float (centred on the centroid), type[n], bonds[n-1][2],
 *   frag[n] (0 = root fragment, k+1 = child fragment of torsion k),
 *   tor_a/tor_b[T] (axis a->b, a on the root side), tor_parent[T] (-1 = root; parents first).
 */
int ligand_gen_one(uint64_t seed, uint64_t index, int n, int t_req, int n_types, int backbone,
                   float* xyz, uint8_t* type, uint8_t* bonds, uint8_t* frag,
                   uint8_t* tor_a, uint8_t* tor_b, int8_t* tor_parent, int* t_out) {
    if (n < 2 || n > MAXN || n_types < 1 || backbone > n) return -1;
    rng_t rng; rng.s = seed * 0xD1342543DE82EF95ULL + index * 0x9E3779B97F4A7C15ULL + 0x1234567ULL;
    rng_next(&rng);
    double x[MAXN][3];
    int deg[MAXN], nbr[MAXN][4];

    for (int attempt = 0; attempt < 200; ++attempt) {
        int ok = 1;
        memset(deg, 0, sizeof(deg));
        x[0][0] = x[0][1] = x[0][2] = 0.0;
        int placed = 1;
        while (placed < n && ok) {
            int done = 0;
            for (int tries = 0; tries < 1000 && !done; ++tries) {
                int p;
                if (placed < backbone) p = placed - 1;                    /* linear chain */
                else { p = rng_int(&rng, placed); if (deg[p] >= 4) continue; }
                double dirs[4][3], d[3];
                for (int k = 0; k < deg[p]; ++k) {
                    for (int c = 0; c < 3; ++c) dirs[k][c] = x[nbr[p][k]][c] - x[p][c];
                    unit3(dirs[k]);
                }
                new_direction(&rng, deg[p], dirs, d);
                double q[3] = {x[p][0] + BOND * d[0], x[p][1] + BOND * d[1], x[p][2] + BOND * d[2]};
                int clash = 0;
                for (int a = 0; a < placed && !clash; ++a) {
                    if (a == p) continue;
                    double dx = q[0] - x[a][0], dy = q[1] - x[a][1], dz = q[2] - x[a][2];
                    if (dx * dx + dy * dy + dz * dz < MIN_NB * MIN_NB) clash = 1;
                }
                if (clash) continue;
                memcpy(x[placed], q, sizeof(q));
                nbr[p][deg[p]++] = placed;
                nbr[placed][0] = p; deg[placed] = 1;
                bonds[2 * (placed - 1)] = (uint8_t)p;
                bonds[2 * (placed - 1) + 1] = (uint8_t)placed;
                ++placed; done = 1;
            }
            if (!done) ok = 0;
        }
        if (!ok) continue;

        /* centre on the centroid, types */
        double c[3] = {0, 0, 0};
        for (int a = 0; a < n; ++a) for (int k = 0; k < 3; ++k) c[k] += x[a][k];
        for (int k = 0; k < 3; ++k) c[k] /= n;
        for (int a = 0; a < n; ++a) {
            for (int k = 0; k < 3; ++k) xyz[3 * a + k] = (float)(x[a][k] - c[k]);
            type[a] = (uint8_t)rng_int(&rng, n_types);
        }

        /* rotatable bonds */
        int nb = n - 1, cand[MAXN], ncand = 0, rot[MAXN];
        memset(rot, 0, sizeof(rot));
        if (backbone > 0) {
            int mid = backbone / 2;
            /* interior backbone bonds (i, i+1), i = 1..backbone-3, nearest the middle first */
            int lo = mid - 1, hi = mid;              /* bond index i joins atoms i and i+1 */
            while (ncand < t_req && (lo >= 1 || hi <= backbone - 3)) {
                if (hi <= backbone - 3 && ncand < t_req) cand[ncand++] = hi++;
                if (lo >= 1 && ncand < t_req) cand[ncand++] = lo--;
            }
            for (int i = 0; i < ncand; ++i) rot[cand[i]] = 1;   /* bond i is bonds[i] = (i, i+1) in chain mode */
        } else {
            for (int b = 0; b < nb; ++b)
                if (deg[bonds[2 * b]] >= 2 && deg[bonds[2 * b + 1]] >= 2) cand[ncand++] = b;
            int t = t_req < ncand ? t_req : ncand;
            for (int i = 0; i < t; ++i) {            /* partial Fisher-Yates */
                int j = i + rng_int(&rng, ncand - i);
                int tmp = cand[i]; cand[i] = cand[j]; cand[j] = tmp;
                rot[cand[i]] = 1;
            }
        }

        /* rigid fragments = components of the tree minus the rotatable bonds */
        int comp[MAXN];
        for (int a = 0; a < n; ++a) comp[a] = -1;
        int ncomp = 0, stack[MAXN];
        for (int a0 = 0; a0 < n; ++a0) {
            if (comp[a0] >= 0) continue;
            int sp = 0; stack[sp++] = a0; comp[a0] = ncomp;
            while (sp) {
                int a = stack[--sp];
                for (int b = 0; b < nb; ++b) {
                    if (rot[b]) continue;
                    int u = bonds[2 * b], v = bonds[2 * b + 1], o = -1;
                    if (u == a) o = v; else if (v == a) o = u;
                    if (o >= 0 && comp[o] < 0) { comp[o] = ncomp; stack[sp++] = o; }
                }
            }
            ++ncomp;
        }
        /* root = fragment of the atom nearest the centroid (G10), or the backbone middle */
        int root_atom = 0;
        if (backbone > 0) root_atom = backbone / 2;
        else {
            double best = 1e30;
            for (int a = 0; a < n; ++a) {
                double d2 = 0; for (int k = 0; k < 3; ++k) d2 += (double)xyz[3 * a + k] * xyz[3 * a + k];
                if (d2 < best) { best = d2; root_atom = a; }
            }
        }
        /* breadth-first walk over fragments: numbers torsions parents-first */
        int label[MAXN], queue[MAXN], qh = 0, qt = 0, via[MAXN], T = 0;
        for (int f = 0; f < ncomp; ++f) label[f] = -1;
        label[comp[root_atom]] = 0; via[comp[root_atom]] = -1; queue[qt++] = comp[root_atom];
        while (qh < qt) {
            int f = queue[qh++];
            for (int b = 0; b < nb; ++b) {
                if (!rot[b]) continue;
                int u = bonds[2 * b], v = bonds[2 * b + 1], a_, b_;
                if (comp[u] == f && label[comp[v]] < 0) { a_ = u; b_ = v; }
                else if (comp[v] == f && label[comp[u]] < 0) { a_ = v; b_ = u; }
                else continue;
                tor_a[T] = (uint8_t)a_; tor_b[T] = (uint8_t)b_;
                tor_parent[T] = (int8_t)via[f];
                label[comp[b_]] = T + 1; via[comp[b_]] = T;
                queue[qt++] = comp[b_];
                ++T;
            }
        }
        for (int a = 0; a < n; ++a) frag[a] = (uint8_t)label[comp[a]];
        *t_out = T;
        return 0;
    }
    return -2;
}

/* Batch: CSR offsets are inputs (atom_off from n[], tor_off sized by t_req[]); writes t_out[]. */
int ligand_gen_batch(uint64_t seed, int n_lig, const int* n, const int* t_req, int n_types, int backbone,
                     const int* atom_off, const int* tor_cap_off,
                     float* xyz, uint8_t* type, uint8_t* bonds /* at 2*(atom_off[i]-i) */, uint8_t* frag,
                     uint8_t* tor_a, uint8_t* tor_b, int8_t* tor_parent, int* t_out) {
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(| : fail)
    for (int i = 0; i < n_lig; ++i) {
        int ao = atom_off[i], to = tor_cap_off[i];
        int rc = ligand_gen_one(seed, (uint64_t)i, n[i], t_req[i], n_types, backbone,
                                xyz + 3 * (size_t)ao, type + ao, bonds + 2 * (size_t)(ao - i), frag + ao,
                                tor_a + to, tor_b + to, tor_parent + to, t_out + i);
        if (rc != 0) fail |= 1;
    }
    return fail ? -1 : 0;
}
