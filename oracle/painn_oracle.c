/*
 * painn_oracle.c -- fp64 CPU ORACLE for the PaiNN energy / force / virial hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_2506_04055_b200/) may import, link or
 * call this file; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs use it.  It shares no code with the CUDA path.  Plain loops, fp64 everywhere, brute-force O(N^2)
 * neighbour search, hand-derived adjoint written exactly in the order of SURVEY.md §8(c) (the reading of
 * the model this build fixes; the paper itself names PaiNN only at PAPER.md:212, 246 and frames the
 * computation by Eq. 1/5, the local-only energy sum, the force sum rule
 * and the message/update form Eq. 6-7).
 *
 * Value-level parity with the paper is UNPINNED (the paper prints no worked number for this path); the
 * oracle is pinned structurally by tests/test_oracle_pins.py (finite differences, an independent
 * dense-autograd restatement, invariances, closed forms, extensivity, ghost == periodic).
 *
 * Build:  gcc -O2 -fopenmp -ffp-contract=off -fPIC -shared painn_oracle.c -o libpainn_oracle.so -lm
 * (-ffp-contract=off: the cutoff predicate must be evaluated without FMA contraction, A4.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define MAXT 8
static const double PI = 3.14159265358979323846;

typedef struct {
    const double *Wm1, *bm1, *Wm2, *bm2, *Wf, *bf, *U, *V, *Wu1, *bu1, *Wu2, *bu2;
} Layer;
typedef struct {
    int n_species, F, K, T, R;
    double rc, eps;
    const double *Emb;
    Layer L[MAXT];
    const double *Wr1, *br1, *wr2, *br2;
} Model;

/* Weight blob layout: SURVEY.md §8(b); header 48 bytes then fp64 arrays in blob order. */
static int parse_blob(const void *blob, size_t nbytes, Model *m) {
    const unsigned char *b = (const unsigned char *)blob;
    if (nbytes < 48 || memcmp(b, "PNN1", 4) != 0) return 2;
    uint32_t h[7];
    memcpy(h, b + 4, sizeof h);
    if (h[0] != 1) return 2;
    m->n_species = (int)h[1]; m->F = (int)h[2]; m->K = (int)h[3]; m->T = (int)h[4]; m->R = (int)h[5];
    memcpy(&m->rc, b + 32, 8);
    memcpy(&m->eps, b + 40, 8);
    if (m->T < 1 || m->T > MAXT || m->F < 1 || m->K < 1 || m->R < 1) return 2;
    const double *p = (const double *)(b + 48);
    size_t F = m->F, K = m->K, R = m->R;
    m->Emb = p; p += (size_t)m->n_species * F;
    for (int t = 0; t < m->T; t++) {
        Layer *l = &m->L[t];
        l->Wm1 = p; p += F * F;       l->bm1 = p; p += F;
        l->Wm2 = p; p += 3 * F * F;   l->bm2 = p; p += 3 * F;
        l->Wf  = p; p += 3 * F * K;   l->bf  = p; p += 3 * F;
        l->U   = p; p += F * F;       l->V   = p; p += F * F;
        l->Wu1 = p; p += F * 2 * F;   l->bu1 = p; p += F;
        l->Wu2 = p; p += 3 * F * F;   l->bu2 = p; p += 3 * F;
    }
    m->Wr1 = p; p += R * F; m->br1 = p; p += R; m->wr2 = p; p += R; m->br2 = p; p += 1;
    if ((size_t)((const unsigned char *)p - b) != nbytes) return 2;
    return 0;
}

static inline double sigmoid(double x) { return 1.0 / (1.0 + exp(-x)); }
static inline double silu(double x) { return x * sigmoid(x); }
/* SiLU'(x) = sigma(x) (1 + x (1 - sigma(x))) */
static inline double dsilu(double x) { double s = sigmoid(x); return s * (1.0 + x * (1.0 - s)); }

/* ------------------------------------------------------------------------------------------------
 * Neighbour set -- the DEFINITION (SURVEY.md §8(c) "Neighbour set"; PAPER.md:68 cutoff pruning).
 * Periodic mode: every ordered pair (i, j) and image S in {-smax..smax}^3 with (i != j or S != 0);
 *   r_e = (r_j + S*L) - r_i from the positions AS GIVEN; edge iff (dx*dx + dy*dy) + dz*dz < rc*rc.
 * Open mode (periodic == 0): all ordered pairs i != j, S = 0.
 * Edges are emitted sorted by (i, j, Sx, Sy, Sz).  Two passes: count rows, then fill.
 * Returns 0, or 1 if cap is too small (n_edges still set to the required count).
 * ---------------------------------------------------------------------------------------------- */
static inline int edge_test(const double *pos, long long i, long long j, const double *box, int sx, int sy,
                            int sz, double rc2, double *r) {
    double dx = (pos[3 * j + 0] + sx * box[0]) - pos[3 * i + 0];
    double dy = (pos[3 * j + 1] + sy * box[1]) - pos[3 * i + 1];
    double dz = (pos[3 * j + 2] + sz * box[2]) - pos[3 * i + 2];
    double d2 = (dx * dx + dy * dy) + dz * dz;
    if (r) { r[0] = dx; r[1] = dy; r[2] = dz; }
    return d2 < rc2;
}

int oracle_neighbors(const double *pos, long long N, const double *box, int periodic, double rc, int smax,
                     long long cap, long long *n_edges, int *ei, int *ej, signed char *img) {
    const double rc2 = rc * rc;
    const int sm = periodic ? smax : 0;
    long long *row = (long long *)calloc((size_t)N + 1, sizeof(long long));
    if (!row) return 5;
#pragma omp parallel for schedule(dynamic, 16)
    for (long long i = 0; i < N; i++) {
        long long c = 0;
        for (long long j = 0; j < N; j++)
            for (int sx = -sm; sx <= sm; sx++)
                for (int sy = -sm; sy <= sm; sy++)
                    for (int sz = -sm; sz <= sm; sz++) {
                        if (i == j && sx == 0 && sy == 0 && sz == 0) continue;
                        c += edge_test(pos, i, j, box, sx, sy, sz, rc2, NULL);
                    }
        row[i + 1] = c;
    }
    for (long long i = 0; i < N; i++) row[i + 1] += row[i];
    *n_edges = row[N];
    if (row[N] > cap) { free(row); return 1; }
#pragma omp parallel for schedule(dynamic, 16)
    for (long long i = 0; i < N; i++) {
        long long e = row[i];
        for (long long j = 0; j < N; j++)
            for (int sx = -sm; sx <= sm; sx++)
                for (int sy = -sm; sy <= sm; sy++)
                    for (int sz = -sm; sz <= sm; sz++) {
                        if (i == j && sx == 0 && sy == 0 && sz == 0) continue;
                        if (edge_test(pos, i, j, box, sx, sy, sz, rc2, NULL)) {
                            ei[e] = (int)i; ej[e] = (int)j;
                            img[3 * e + 0] = (signed char)sx; img[3 * e + 1] = (signed char)sy;
                            img[3 * e + 2] = (signed char)sz;
                            e++;
                        }
                    }
    }
    free(row);
    return 0;
}

/* y[out] = W[out x in] x + b */
static void matvec(const double *W, const double *b, const double *x, double *y, int out, int in) {
    for (int o = 0; o < out; o++) {
        double a = b ? b[o] : 0.0;
        const double *w = W + (size_t)o * in;
        for (int k = 0; k < in; k++) a += w[k] * x[k];
        y[o] = a;
    }
}
/* x[in] += W^T y  (W is [out x in]) */
static void matvec_T_acc(const double *W, const double *y, double *x, int out, int in) {
    for (int o = 0; o < out; o++) {
        const double *w = W + (size_t)o * in;
        double yo = y[o];
        for (int k = 0; k < in; k++) x[k] += w[k] * yo;
    }
}

/* Radial basis and cutoff (SURVEY.md §8(c) Forward, readings A3/A5):
 *   rho_n(d) = sin(n pi d / rc) / d, n = 1..K;  fc(d) = (1 + cos(pi d / rc)) / 2
 *   rho'_n = (n pi / rc) cos(n pi d / rc) / d - sin(n pi d / rc) / d^2;  fc' = -(pi / 2 rc) sin(pi d / rc) */
static void radial(double d, double rc, int K, double *rho, double *drho, double *fc, double *dfc) {
    for (int n = 1; n <= K; n++) {
        double a = n * PI / rc;
        rho[n - 1] = sin(a * d) / d;
        if (drho) drho[n - 1] = a * cos(a * d) / d - sin(a * d) / (d * d);
    }
    *fc = 0.5 * (1.0 + cos(PI * d / rc));
    if (dfc) *dfc = -(PI / (2.0 * rc)) * sin(PI * d / rc);
}

typedef struct {
    double *s_in, *v_in;   /* layer inputs            [N*F], [N*3*F] */
    double *hpre, *phi;    /* Wm1 s + bm1 [N*F];  phi [N*3F] = [s | vs | vv] */
    double *s1, *v1;       /* s', v' after message    */
    double *p, *q, *nrm;   /* U v', V v' [N*3*F]; n [N*F] */
    double *zpre, *a;      /* Wu1[s';n]+bu1 [N*F];  a [N*3F] = [vv | sv | ss] */
} Saved;

static double *dalloc(size_t n) { return (double *)calloc(n ? n : 1, sizeof(double)); }

/*
 * oracle_compute -- E = sum_{i<n_local} E_i, F = -dE/dr, virial W_ab = -sum_e r_e,a g_e,b.
 *   periodic != 0: minimum-image style periodic graph over the N = n_local + n_ghost atoms in `box`
 *   periodic == 0: open boundaries (ghost mode; the ghosts ARE the periodicity)
 *   ghost_owner (may be NULL): fold F_ghost onto F_owner and zero the ghost row
 *   virial: 6 components xx,yy,zz,xy,xz,yz (off-diagonals averaged); virial9 (may be NULL): raw 3x3 W_ab
 *   atom_energy (may be NULL): E_i for all N atoms
 *   state_dump (may be NULL): [(T+1) x N x 4F] layer states (s | v_x | v_y | v_z) after embed and each layer
 *   n_edges_out (may be NULL)
 * Returns 0 on success (error codes follow include/mlp.h numbering).
 */
int oracle_compute(const void *blob, size_t nbytes, const double *pos, const int *types, const double *box,
                   long long n_local, long long n_ghost, int periodic, int smax, const int *ghost_owner,
                   double *energy, double *forces, double *virial, double *virial9, double *atom_energy,
                   double *state_dump, long long *n_edges_out) {
    Model M;
    int rcode = parse_blob(blob, nbytes, &M);
    if (rcode) return rcode;
    const long long N = n_local + n_ghost;
    const int F = M.F, K = M.K, T = M.T, R = M.R;
    const size_t F3 = 3 * (size_t)F;
    for (long long i = 0; i < N; i++)
        if (types[i] < 0 || types[i] >= M.n_species) return 4;

    /* ---- neighbour list (brute force) ---- */
    long long E = 0;
    oracle_neighbors(pos, N, box, periodic, M.rc, smax, 0, &E, NULL, NULL, NULL);
    int *ei = (int *)malloc(sizeof(int) * (size_t)(E ? E : 1));
    int *ej = (int *)malloc(sizeof(int) * (size_t)(E ? E : 1));
    signed char *img = (signed char *)malloc(3 * (size_t)(E ? E : 1));
    if (!ei || !ej || !img) return 5;
    rcode = oracle_neighbors(pos, N, box, periodic, M.rc, smax, E, &E, ei, ej, img);
    if (rcode) return rcode;
    if (n_edges_out) *n_edges_out = E;

    /* row pointers by receiver (edges are sorted by i) and an index sorted by sender j */
    long long *rowp = (long long *)calloc((size_t)N + 1, sizeof(long long));
    long long *colp = (long long *)calloc((size_t)N + 2, sizeof(long long));
    long long *by_sender = (long long *)malloc(sizeof(long long) * (size_t)(E ? E : 1));
    for (long long e = 0; e < E; e++) { rowp[ei[e] + 1]++; colp[ej[e] + 2]++; }
    for (long long i = 0; i < N; i++) { rowp[i + 1] += rowp[i]; colp[i + 2] += colp[i + 1]; }
    for (long long e = 0; e < E; e++) by_sender[colp[ej[e] + 1]++] = e;   /* colp[j] .. colp[j+1] afterwards */

    /* per-edge geometry: r_e = r_j + S L - r_i, d, u = r_e / d */
    double *re = dalloc(3 * (size_t)E), *de = dalloc((size_t)E), *ge = dalloc(3 * (size_t)E);
    for (long long e = 0; e < E; e++) {
        double r[3];
        edge_test(pos, ei[e], ej[e], box, img[3 * e], img[3 * e + 1], img[3 * e + 2], 0.0, r);
        re[3 * e] = r[0]; re[3 * e + 1] = r[1]; re[3 * e + 2] = r[2];
        de[e] = sqrt((r[0] * r[0] + r[1] * r[1]) + r[2] * r[2]);
    }

    /* ---- forward ---- */
    double *s = dalloc((size_t)N * F), *v = dalloc((size_t)N * F3);
    for (long long i = 0; i < N; i++)
        for (int f = 0; f < F; f++) s[i * F + f] = M.Emb[(size_t)types[i] * F + f];   /* s0 = Emb[z], v0 = 0 */
    if (state_dump) {
        for (long long i = 0; i < N; i++) {
            memcpy(state_dump + (size_t)i * 4 * F, s + i * F, sizeof(double) * F);
            memcpy(state_dump + (size_t)i * 4 * F + F, v + i * F3, sizeof(double) * F3);
        }
    }
    Saved *S = (Saved *)calloc((size_t)T, sizeof(Saved));
    for (int t = 0; t < T; t++) {
        const Layer *l = &M.L[t];
        Saved *sv = &S[t];
        sv->s_in = dalloc((size_t)N * F); sv->v_in = dalloc((size_t)N * F3);
        sv->hpre = dalloc((size_t)N * F); sv->phi = dalloc((size_t)N * F3);
        sv->s1 = dalloc((size_t)N * F); sv->v1 = dalloc((size_t)N * F3);
        sv->p = dalloc((size_t)N * F3); sv->q = dalloc((size_t)N * F3); sv->nrm = dalloc((size_t)N * F);
        sv->zpre = dalloc((size_t)N * F); sv->a = dalloc((size_t)N * F3);
        memcpy(sv->s_in, s, sizeof(double) * (size_t)N * F);
        memcpy(sv->v_in, v, sizeof(double) * (size_t)N * F3);
        /* h_j = SiLU(Wm1 s_j + bm1);  phi_j = Wm2 h_j + bm2 */
#pragma omp parallel
        {
            double *h = dalloc(F);
#pragma omp for schedule(static)
            for (long long j = 0; j < N; j++) {
                matvec(l->Wm1, l->bm1, s + j * F, sv->hpre + j * F, F, F);
                for (int f = 0; f < F; f++) h[f] = silu(sv->hpre[j * F + f]);
                matvec(l->Wm2, l->bm2, h, sv->phi + j * F3, 3 * F, F);
            }
            free(h);
        }
        /* messages: s'_i = s_i + sum_e w^s o phi^s_j ; v'_i[c] = v_i[c] + sum_e (w^vs o phi^vs_j u[c] + w^vv o phi^vv_j o v_j[c]) */
#pragma omp parallel
        {
            double *rho = dalloc(K), *w = dalloc(F3);
#pragma omp for schedule(dynamic, 8)
            for (long long i = 0; i < N; i++) {
                double *s1 = sv->s1 + i * F, *v1 = sv->v1 + i * F3;
                for (int f = 0; f < F; f++) s1[f] = s[i * F + f];
                for (size_t f = 0; f < F3; f++) v1[f] = v[i * F3 + f];
                for (long long e = rowp[i]; e < rowp[i + 1]; e++) {
                    long long j = ej[e];
                    double d = de[e], fc, u[3] = {re[3 * e] / d, re[3 * e + 1] / d, re[3 * e + 2] / d};
                    radial(d, M.rc, K, rho, NULL, &fc, NULL);
                    matvec(l->Wf, l->bf, rho, w, 3 * F, K);
                    for (size_t f = 0; f < F3; f++) w[f] *= fc;            /* w = fc (Wf rho + bf), A5 */
                    const double *ph = sv->phi + j * F3, *vj = v + j * F3;
                    for (int f = 0; f < F; f++) {
                        s1[f] += w[f] * ph[f];
                        double xvs = w[F + f] * ph[F + f], xvv = w[2 * F + f] * ph[2 * F + f];
                        for (int c = 0; c < 3; c++) v1[c * F + f] += xvs * u[c] + xvv * vj[c * F + f];
                    }
                }
            }
            free(rho); free(w);
        }
        /* update */
#pragma omp parallel
        {
            double *sn = dalloc(2 * F), *g = dalloc(F);
#pragma omp for schedule(static)
            for (long long i = 0; i < N; i++) {
                const double *s1 = sv->s1 + i * F, *v1 = sv->v1 + i * F3;
                double *p = sv->p + i * F3, *q = sv->q + i * F3, *nr = sv->nrm + i * F, *a = sv->a + i * F3;
                for (int c = 0; c < 3; c++) {
                    matvec(l->U, NULL, v1 + c * F, p + c * F, F, F);
                    matvec(l->V, NULL, v1 + c * F, q + c * F, F, F);
                }
                for (int f = 0; f < F; f++) {
                    nr[f] = sqrt(q[f] * q[f] + q[F + f] * q[F + f] + q[2 * F + f] * q[2 * F + f] + M.eps);
                    sn[f] = s1[f]; sn[F + f] = nr[f];
                }
                matvec(l->Wu1, l->bu1, sn, sv->zpre + i * F, F, 2 * F);
                for (int f = 0; f < F; f++) g[f] = silu(sv->zpre[i * F + f]);
                matvec(l->Wu2, l->bu2, g, a, 3 * F, F);                    /* a = [vv | sv | ss] */
                for (int f = 0; f < F; f++) {
                    double D = p[f] * q[f] + p[F + f] * q[F + f] + p[2 * F + f] * q[2 * F + f];
                    for (int c = 0; c < 3; c++) v[i * F3 + c * F + f] = v1[c * F + f] + a[f] * p[c * F + f];
                    s[i * F + f] = s1[f] + a[F + f] * D + a[2 * F + f];
                }
            }
            free(sn); free(g);
        }
        if (state_dump) {
            double *dst = state_dump + (size_t)(t + 1) * N * 4 * F;
            for (long long i = 0; i < N; i++) {
                memcpy(dst + (size_t)i * 4 * F, s + i * F, sizeof(double) * F);
                memcpy(dst + (size_t)i * 4 * F + F, v + i * F3, sizeof(double) * F3);
            }
        }
    }
    /* readout: E_i = wr2 . SiLU(Wr1 s_i + br1) + br2 ;  E = sum over LOCAL atoms */
    double *rpre = dalloc((size_t)N * R), *Ei = dalloc((size_t)N);
    double Etot = 0.0;
    for (long long i = 0; i < N; i++) {
        matvec(M.Wr1, M.br1, s + i * F, rpre + i * R, R, F);
        double a = M.br2[0];
        for (int r = 0; r < R; r++) a += M.wr2[r] * silu(rpre[i * R + r]);
        Ei[i] = a;
        if (i < n_local) Etot += a;
    }
    if (atom_energy) memcpy(atom_energy, Ei, sizeof(double) * (size_t)N);

    /* ---- adjoint (xb == dE/dx) ---- */
    double *sb = dalloc((size_t)N * F), *vb = dalloc((size_t)N * F3);
    for (long long i = 0; i < n_local; i++) {           /* sb_i = [i local] Wr1^T (wr2 o SiLU'(.)) ; vb = 0 */
        double *tmp = dalloc(R);
        for (int r = 0; r < R; r++) tmp[r] = M.wr2[r] * dsilu(rpre[i * R + r]);
        matvec_T_acc(M.Wr1, tmp, sb + i * F, R, F);
        free(tmp);
    }
    double *s1b = dalloc((size_t)N * F), *v1b = dalloc((size_t)N * F3);
    double *phib = dalloc((size_t)N * F3);
    for (int t = T - 1; t >= 0; t--) {
        const Layer *l = &M.L[t];
        const Saved *sv = &S[t];
        /* update adjoint, per atom: produces s1b (= sb'), v1b (= vb') */
#pragma omp parallel
        {
            double *ab = dalloc(F3), *pb = dalloc(F3), *qb = dalloc(F3), *gb = dalloc(F), *zb = dalloc(F),
                   *snb = dalloc(2 * F);
#pragma omp for schedule(static)
            for (long long i = 0; i < N; i++) {
                const double *p = sv->p + i * F3, *q = sv->q + i * F3, *a = sv->a + i * F3, *nr = sv->nrm + i * F;
                const double *sbi = sb + i * F, *vbi = vb + i * F3;
                for (int f = 0; f < F; f++) {
                    double D = p[f] * q[f] + p[F + f] * q[F + f] + p[2 * F + f] * q[2 * F + f];
                    double Db = sbi[f] * a[F + f];                                      /* Db = sb o a^sv */
                    ab[f] = vbi[f] * p[f] + vbi[F + f] * p[F + f] + vbi[2 * F + f] * p[2 * F + f];
                    ab[F + f] = sbi[f] * D;
                    ab[2 * F + f] = sbi[f];
                    for (int c = 0; c < 3; c++) {
                        pb[c * F + f] = vbi[c * F + f] * a[f] + Db * q[c * F + f];
                        qb[c * F + f] = Db * p[c * F + f];
                    }
                }
                memset(gb, 0, sizeof(double) * F);
                matvec_T_acc(l->Wu2, ab, gb, 3 * F, F);
                for (int f = 0; f < F; f++) zb[f] = gb[f] * dsilu(sv->zpre[i * F + f]);
                memset(snb, 0, sizeof(double) * 2 * F);
                matvec_T_acc(l->Wu1, zb, snb, F, 2 * F);                               /* [ds ; nb] */
                for (int f = 0; f < F; f++)
                    for (int c = 0; c < 3; c++) qb[c * F + f] += snb[F + f] * q[c * F + f] / nr[f];
                for (int f = 0; f < F; f++) s1b[i * F + f] = sbi[f] + snb[f];
                for (int c = 0; c < 3; c++) {
                    double *o = v1b + i * F3 + c * F;
                    for (int f = 0; f < F; f++) o[f] = vbi[c * F + f];
                    matvec_T_acc(l->U, pb + c * F, o, F, F);
                    matvec_T_acc(l->V, qb + c * F, o, F, F);
                }
            }
            free(ab); free(pb); free(qb); free(gb); free(zb); free(snb);
        }
        /* message adjoint: residual path, then every edge e = (i <- j) scatters onto its sender j.
           The loop runs sender by sender (by_sender index) so each thread owns phib_j, vb_j, g_e. */
        memcpy(sb, s1b, sizeof(double) * (size_t)N * F);
        memcpy(vb, v1b, sizeof(double) * (size_t)N * F3);
        memset(phib, 0, sizeof(double) * (size_t)N * F3);
#pragma omp parallel
        {
            double *rho = dalloc(K), *drho = dalloc(K), *lin = dalloc(F3), *w = dalloc(F3), *wb = dalloc(F3),
                   *wfT = dalloc(K);
#pragma omp for schedule(dynamic, 8)
            for (long long j = 0; j < N; j++) {
                const double *ph = sv->phi + j * F3, *vj = sv->v_in + j * F3;
                for (long long x = colp[j]; x < colp[j + 1]; x++) {
                    long long e = by_sender[x], i = ei[e];
                    double d = de[e], fc, dfc, u[3] = {re[3 * e] / d, re[3 * e + 1] / d, re[3 * e + 2] / d};
                    radial(d, M.rc, K, rho, drho, &fc, &dfc);
                    matvec(l->Wf, l->bf, rho, lin, 3 * F, K);                           /* lin = Wf rho + bf */
                    for (size_t f = 0; f < F3; f++) w[f] = fc * lin[f];
                    const double *si = s1b + i * F, *vi = v1b + i * F3;
                    double ub[3] = {0, 0, 0};
                    for (int f = 0; f < F; f++) {
                        double X = vi[f] * u[0] + vi[F + f] * u[1] + vi[2 * F + f] * u[2];
                        double Z = vi[f] * vj[f] + vi[F + f] * vj[F + f] + vi[2 * F + f] * vj[2 * F + f];
                        phib[j * F3 + f] += w[f] * si[f];
                        phib[j * F3 + F + f] += w[F + f] * X;
                        phib[j * F3 + 2 * F + f] += w[2 * F + f] * Z;
                        for (int c = 0; c < 3; c++) {
                            vb[j * F3 + c * F + f] += w[2 * F + f] * ph[2 * F + f] * vi[c * F + f];
                            ub[c] += w[F + f] * ph[F + f] * vi[c * F + f];
                        }
                        wb[f] = ph[f] * si[f];
                        wb[F + f] = ph[F + f] * X;
                        wb[2 * F + f] = ph[2 * F + f] * Z;
                    }
                    /* db = fc' sum_f wb (Wf rho + bf) + fc sum_n rho'_n (Wf^T wb)_n */
                    double db = 0.0, t1 = 0.0;
                    for (size_t f = 0; f < F3; f++) t1 += wb[f] * lin[f];
                    memset(wfT, 0, sizeof(double) * K);
                    matvec_T_acc(l->Wf, wb, wfT, 3 * F, K);
                    for (int n = 0; n < K; n++) db += drho[n] * wfT[n];
                    db = dfc * t1 + fc * db;
                    double uu = ub[0] * u[0] + ub[1] * u[1] + ub[2] * u[2];
                    for (int c = 0; c < 3; c++) ge[3 * e + c] += db * u[c] + (ub[c] - uu * u[c]) / d;
                }
            }
            free(rho); free(drho); free(lin); free(w); free(wb); free(wfT);
        }
        /* phi-MLP adjoint: sb_j += Wm1^T ((Wm2^T phib_j) o SiLU'(hpre_j)) */
#pragma omp parallel
        {
            double *hb = dalloc(F);
#pragma omp for schedule(static)
            for (long long j = 0; j < N; j++) {
                memset(hb, 0, sizeof(double) * F);
                matvec_T_acc(l->Wm2, phib + j * F3, hb, 3 * F, F);
                for (int f = 0; f < F; f++) hb[f] *= dsilu(sv->hpre[j * F + f]);
                matvec_T_acc(l->Wm1, hb, sb + j * F, F, F);
            }
            free(hb);
        }
    }

    /* ---- forces, virial, ghost fold ---- */
    double W[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    memset(forces, 0, sizeof(double) * 3 * (size_t)N);
    for (long long e = 0; e < E; e++) {
        for (int c = 0; c < 3; c++) {
            forces[3 * (size_t)ej[e] + c] -= ge[3 * e + c];     /* sender:   dE/dr_j = +g_e */
            forces[3 * (size_t)ei[e] + c] += ge[3 * e + c];     /* receiver: dE/dr_i = -g_e */
            for (int b = 0; b < 3; b++) W[3 * c + b] -= re[3 * e + c] * ge[3 * e + b];
        }
    }
    if (ghost_owner) {
        for (long long g = 0; g < n_ghost; g++) {
            long long o = ghost_owner[g];
            for (int c = 0; c < 3; c++) {
                forces[3 * o + c] += forces[3 * (n_local + g) + c];
                forces[3 * (n_local + g) + c] = 0.0;
            }
        }
    }
    *energy = Etot;
    virial[0] = W[0]; virial[1] = W[4]; virial[2] = W[8];
    virial[3] = 0.5 * (W[1] + W[3]); virial[4] = 0.5 * (W[2] + W[6]); virial[5] = 0.5 * (W[5] + W[7]);
    if (virial9) memcpy(virial9, W, sizeof W);

    for (int t = 0; t < T; t++) {
        Saved *sv = &S[t];
        free(sv->s_in); free(sv->v_in); free(sv->hpre); free(sv->phi); free(sv->s1); free(sv->v1);
        free(sv->p); free(sv->q); free(sv->nrm); free(sv->zpre); free(sv->a);
    }
    free(S); free(s); free(v); free(sb); free(vb); free(s1b); free(v1b); free(phib); free(rpre); free(Ei);
    free(re); free(de); free(ge); free(rowp); free(colp); free(by_sender); free(ei); free(ej); free(img);
    return 0;
}

/* number of OpenMP threads the oracle will use (reported by bench.py's cpu_baseline) */
int oracle_threads(void) {
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
