/*
 * ORACLE (test infrastructure, not product code).  Plain, slow, obviously-correct CPU
 * implementation of what the hot path computes.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call this.  It shares no code
 * with the CUDA path (paper_2311_02854_b200/csrc); only array formats are common.
 *
 * Tier O-pair  (opair_sigma):  sigma = H psi by the operator-pair contraction,
 *   sigma[qL',c1',c2',qR'] += c_mu * zeta * o1[c1',c1] * o2[c2',c2]
 *                             * O^L[qL',qL] * psi[qL,c1,c2,qR] * (O^R[qR',qR])^T
 *   PAPER.md:68-71 (Eq. 7), PAPER.md:89-93 (Eqs. 11-13); zeta = DESIGN.md reading 3:
 *   (-1)^{ p_C1 N_l + p_C2 (N_l+N_c1) + p_R (N_l+N_c1+N_c2) } from the ket quantum numbers.
 *   Linear-combination operators ("intermediates") are formed first.
 * Tier O-def   (fci_dense_h):  dense determinant-basis H from the Slater-Condon rules
 *   for Eq. (2) -- the plain definition of the exact result.
 * opair_hdiag: the diagonal of the same operator ("diagonal part of
 *   Hamiltonian"), term by term.
 *
 * All arithmetic FP64, plain loops, no blocking, no reordering beyond the formula.
 * OpenMP only distributes independent output blocks (or, for a handful of blocks, independent output rows) over
 * threads; the summation order of every element is fixed.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static const int SITE_N[4] = {0, 1, 1, 2};
static const int SITE_S[4] = {0, -1, 1, 0};

typedef struct {
    const int32_t *secL, *secR;   /* [n][3] N, 2Sz, dim */
    int nsecL, nsecR;
    const int64_t *ops;           /* [nops][8] side kind p q dN d2Sz first nblocks */
    int nops;
    const int64_t *blocks;        /* [nblk][3] row col offset */
    const double *values;
    const int64_t *lin_ptr; const int32_t *lin_op; const double *lin_coef;
    const double *site_ops; const int32_t *site_parity; int nsite;
    const double *term_coef; const int32_t *term_idx; int64_t nterms;
    const int64_t *layout;        /* [nblkpsi][7] iL c1 c2 iR dL dR offset */
    int64_t npsiblk;
} problem_t;

/* per-op dense block table: blk[op][row_sector] -> pointer (or NULL), since charge fixes col */
typedef struct { double **rowblk; int *colsec; int nsec; int parity; } optab_t;

static int sec_find(const int32_t *sec, int n, int N, int S) {
    for (int i = 0; i < n; i++) if (sec[3 * i] == N && sec[3 * i + 1] == S) return i;
    return -1;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* form_values = 0: structure only (which blocks exist); used by opair_count, which needs no arithmetic */
static optab_t *build_optabs(const problem_t *P, double ***owned, int *nowned, int form_values) {
    optab_t *T = (optab_t *)calloc(P->nops, sizeof(optab_t));
    *owned = (double **)calloc(P->nops, sizeof(double *));
    *nowned = 0;
    for (int o = 0; o < P->nops; o++) {
        const int64_t *op = P->ops + 8 * o;
        int side = (int)op[0], kind = (int)op[1];
        const int32_t *sec = side == 0 ? P->secL : P->secR;
        int nsec = side == 0 ? P->nsecL : P->nsecR;
        T[o].nsec = nsec;
        T[o].parity = (int)(op[4] & 1);
        T[o].rowblk = (double **)calloc(nsec, sizeof(double *));
        T[o].colsec = (int *)malloc(nsec * sizeof(int));
        for (int r = 0; r < nsec; r++)
            T[o].colsec[r] = sec_find(sec, nsec, sec[3 * r] - (int)op[4], sec[3 * r + 1] - (int)op[5]);
        if (kind != 7) {
            for (int64_t b = op[6]; b < op[6] + op[7]; b++) {
                const int64_t *bd = P->blocks + 3 * b;
                T[o].rowblk[bd[0]] = form_values ? (double *)(P->values + bd[2]) : (double *)P->values;   /* presence only */
            }
        }
    }
    /* linear combinations: W = sum_s coef_s * op_s, block by block */
    for (int o = 0; o < P->nops; o++) {
        const int64_t *op = P->ops + 8 * o;
        if (op[1] != 7) continue;
        int side = (int)op[0];
        const int32_t *sec = side == 0 ? P->secL : P->secR;
        int nsec = T[o].nsec;
        int64_t j = op[2];
        size_t total = 0;
        for (int r = 0; r < nsec; r++) {
            int c = T[o].colsec[r];
            if (c < 0) continue;
            int has = 0;
            for (int64_t i = P->lin_ptr[j]; i < P->lin_ptr[j + 1]; i++)
                if (T[P->lin_op[i]].rowblk[r]) has = 1;
            if (has) total += (size_t)sec[3 * r + 2] * sec[3 * c + 2];
        }
        double *buf = (double *)calloc(form_values && total ? total : 1, sizeof(double));
        (*owned)[(*nowned)++] = buf;
        size_t off = 0;
        for (int r = 0; r < nsec; r++) {
            int c = T[o].colsec[r];
            if (c < 0) continue;
            size_t n = (size_t)sec[3 * r + 2] * sec[3 * c + 2];
            int has = 0;
            for (int64_t i = P->lin_ptr[j]; i < P->lin_ptr[j + 1]; i++) {
                const double *src = T[P->lin_op[i]].rowblk[r];
                if (!src) continue;
                has = 1;
                if (!form_values) continue;
                double cf = P->lin_coef[i];
                for (size_t e = 0; e < n; e++) buf[off + e] += cf * src[e];
            }
            if (has) { T[o].rowblk[r] = form_values ? buf + off : buf; off += n; }
        }
    }
    return T;
}

static void free_optabs(optab_t *T, int nops, double **owned, int nowned) {
    for (int o = 0; o < nops; o++) { free(T[o].rowblk); free(T[o].colsec); }
    free(T);
    for (int i = 0; i < nowned; i++) free(owned[i]);
    free(owned);
}

typedef struct { int64_t term; int32_t in_blk, out_blk; const double *Lm; int Lt; const double *Rm; int Rt;
                 int dLo, dLi, dRo, dRi; double alpha; } task_t;

/* Enumerate every (term, psi block, dot transition) contribution. */
static task_t *enumerate_tasks(const problem_t *P, const optab_t *T, int64_t *ntask_out,
                               int diag_only) {
    int64_t cap = 1 << 16, n = 0;
    task_t *tasks = (task_t *)malloc(cap * sizeof(task_t));
    /* lookup of psi blocks by (iL,c1,c2,iR) */
    int64_t nl = P->nsecL, nr = P->nsecR;
    int32_t *lut = (int32_t *)malloc(sizeof(int32_t) * nl * 16 * nr);
    for (int64_t i = 0; i < nl * 16 * nr; i++) lut[i] = -1;
    for (int64_t b = 0; b < P->npsiblk; b++) {
        const int64_t *lb = P->layout + 7 * b;
        lut[((lb[0] * 4 + lb[1]) * 4 + lb[2]) * nr + lb[3]] = (int32_t)b;
    }
    for (int64_t t = 0; t < P->nterms; t++) {
        const int32_t *ti = P->term_idx + 6 * t;
        int ol = ti[0], tl = ti[1], s1 = ti[2], s2 = ti[3], orr = ti[4], tr = ti[5];
        const double *o1 = P->site_ops + 16 * s1, *o2 = P->site_ops + 16 * s2;
        int p1 = P->site_parity[s1], p2 = P->site_parity[s2];
        int pR = orr >= 0 ? T[orr].parity : 0;
        for (int64_t b = 0; b < P->npsiblk; b++) {
            const int64_t *lb = P->layout + 7 * b;
            int iL = (int)lb[0], c1 = (int)lb[1], c2 = (int)lb[2], iR = (int)lb[3];
            int Nl = P->secL[3 * iL];
            int zexp = p1 * Nl + p2 * (Nl + SITE_N[c1]) + pR * (Nl + SITE_N[c1] + SITE_N[c2]);
            double zeta = (zexp & 1) ? -1.0 : 1.0;
            /* L factor: normal use maps col sector -> row sector; transposed use maps row -> col */
            int iLo; const double *Lm = NULL;
            if (ol < 0) iLo = iL;
            else if (!tl) {
                iLo = -1;
                for (int r = 0; r < T[ol].nsec; r++)
                    if (T[ol].colsec[r] == iL && T[ol].rowblk[r]) { iLo = r; Lm = T[ol].rowblk[r]; }
            } else {
                iLo = T[ol].rowblk[iL] ? T[ol].colsec[iL] : -1;
                Lm = T[ol].rowblk[iL];
            }
            if (iLo < 0) continue;
            int iRo; const double *Rm = NULL;
            if (orr < 0) iRo = iR;
            else if (!tr) {
                iRo = -1;
                for (int r = 0; r < T[orr].nsec; r++)
                    if (T[orr].colsec[r] == iR && T[orr].rowblk[r]) { iRo = r; Rm = T[orr].rowblk[r]; }
            } else {
                iRo = T[orr].rowblk[iR] ? T[orr].colsec[iR] : -1;
                Rm = T[orr].rowblk[iR];
            }
            if (iRo < 0) continue;
            for (int c1o = 0; c1o < 4; c1o++) {
                double v1 = o1[4 * c1o + c1];
                if (v1 == 0.0) continue;
                for (int c2o = 0; c2o < 4; c2o++) {
                    double v2 = o2[4 * c2o + c2];
                    if (v2 == 0.0) continue;
                    int32_t ob = lut[(((int64_t)iLo * 4 + c1o) * 4 + c2o) * nr + iRo];
                    if (ob < 0) continue;   /* leaves the (N,Sz) block table: cannot happen for neutral terms */
                    if (diag_only && ob != b) continue;
                    if (n == cap) { cap *= 2; tasks = (task_t *)realloc(tasks, cap * sizeof(task_t)); }
                    task_t *k = &tasks[n++];
                    k->term = t; k->in_blk = (int32_t)b; k->out_blk = ob;
                    k->Lm = Lm; k->Lt = tl; k->Rm = Rm; k->Rt = tr;
                    k->dLi = P->secL[3 * iL + 2]; k->dLo = P->secL[3 * iLo + 2];
                    k->dRi = P->secR[3 * iR + 2]; k->dRo = P->secR[3 * iRo + 2];
                    k->alpha = P->term_coef[t] * zeta * v1 * v2;
                }
            }
        }
    }
    free(lut);
    *ntask_out = n;
    return tasks;
}

static problem_t make_problem(const int32_t *secL, int nsecL, const int32_t *secR, int nsecR,
    const int64_t *ops, int nops, const int64_t *blocks, const double *values,
    const int64_t *lin_ptr, const int32_t *lin_op, const double *lin_coef,
    const double *site_ops, const int32_t *site_parity, int nsite,
    const double *term_coef, const int32_t *term_idx, int64_t nterms,
    const int64_t *layout, int64_t npsiblk) {
    problem_t P;
    P.secL = secL; P.nsecL = nsecL; P.secR = secR; P.nsecR = nsecR; P.ops = ops; P.nops = nops;
    P.blocks = blocks; P.values = values; P.lin_ptr = lin_ptr; P.lin_op = lin_op; P.lin_coef = lin_coef;
    P.site_ops = site_ops; P.site_parity = site_parity; P.nsite = nsite;
    P.term_coef = term_coef; P.term_idx = term_idx; P.nterms = nterms; P.layout = layout; P.npsiblk = npsiblk;
    return P;
}

static int cmp_task_out(const void *a, const void *b) {
    const task_t *x = (const task_t *)a, *y = (const task_t *)b;
    if (x->out_blk != y->out_blk) return x->out_blk < y->out_blk ? -1 : 1;
    if (x->term != y->term) return x->term < y->term ? -1 : 1;
    return x->in_blk < y->in_blk ? -1 : (x->in_blk > y->in_blk);
}

/* sigma = H psi.  only_out: optional list of output-block indices to compute (others left 0).
 * flops_out: 2 dLi dRi dRo + 2 dLo dLi dRo summed over executed tasks (PAPER.md:151 cost measure).
 * Returns number of tasks executed. */
int64_t opair_sigma(const int32_t *secL, int nsecL, const int32_t *secR, int nsecR,
    const int64_t *ops, int nops, const int64_t *blocks, const double *values,
    const int64_t *lin_ptr, const int32_t *lin_op, const double *lin_coef,
    const double *site_ops, const int32_t *site_parity, int nsite,
    const double *term_coef, const int32_t *term_idx, int64_t nterms,
    const int64_t *layout, int64_t npsiblk, int64_t psi_size,
    const double *psi, double *sigma, const int32_t *only_out, int n_only, double *flops_out) {
    problem_t P = make_problem(secL, nsecL, secR, nsecR, ops, nops, blocks, values, lin_ptr, lin_op, lin_coef,
                               site_ops, site_parity, nsite, term_coef, term_idx, nterms, layout, npsiblk);
    double **owned; int nowned;
    optab_t *T = build_optabs(&P, &owned, &nowned, 1);
    int64_t ntask;
    task_t *tasks = enumerate_tasks(&P, T, &ntask, 0);
    qsort(tasks, ntask, sizeof(task_t), cmp_task_out);
    char *want = (char *)malloc(npsiblk);
    memset(want, n_only > 0 ? 0 : 1, npsiblk);
    for (int i = 0; i < n_only; i++) want[only_out[i]] = 1;
    int64_t *start = (int64_t *)malloc((npsiblk + 1) * sizeof(int64_t));
    { int64_t k = 0; for (int64_t b = 0; b <= npsiblk; b++) { while (k < ntask && tasks[k].out_blk < b) k++; start[b] = k; } }
    memset(sigma, 0, psi_size * sizeof(double));
    double flops = 0.0; int64_t done = 0;
    /* Threads: whole output blocks are dealt to threads; when only a few blocks are asked for (fewer than threads),
     * the rows i of each product are dealt to threads instead.  Either way every output element is summed by one
     * thread in the same order (tasks in (term, input block) order, kk ascending): the result does not depend on
     * the thread count or on which of the two modes ran. */
    int rows_mode = 0;
#ifdef _OPENMP
    rows_mode = (n_only > 0 && n_only < omp_get_max_threads());
#endif
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : flops, done) if (!rows_mode)
    for (int64_t ob = 0; ob < npsiblk; ob++) {
        if (!want[ob]) continue;
        double *out = sigma + layout[7 * ob + 6];
        for (int64_t k = start[ob]; k < start[ob + 1]; k++) {
            const task_t *t = &tasks[k];
            const double *x = psi + layout[7 * t->in_blk + 6];
            int dLi = t->dLi, dLo = t->dLo, dRi = t->dRi, dRo = t->dRo;
            /* step 1 (Eq. 11): X[i][j] = sum_k psi[i][k] * OR[j][k]   (OR = R block or its transpose) */
            double *X = (double *)calloc((size_t)dLi * dRo, sizeof(double));
            if (!t->Rm) memcpy(X, x, sizeof(double) * dLi * dRi);
            else {
#pragma omp parallel for schedule(static) if (rows_mode && (double)dLi * dRi * dRo > 2e5)
                for (int i = 0; i < dLi; i++)
                    for (int kk = 0; kk < dRi; kk++) {
                        double a = x[(size_t)i * dRi + kk];
                        if (!t->Rt) for (int j = 0; j < dRo; j++) X[(size_t)i * dRo + j] += a * t->Rm[(size_t)j * dRi + kk];
                        else        for (int j = 0; j < dRo; j++) X[(size_t)i * dRo + j] += a * t->Rm[(size_t)kk * dRo + j];
                    }
                flops += 2.0 * dLi * dRi * dRo;
            }
            /* step 2 + reduction (Eqs. 12-13): sigma[i][j] += alpha * sum_k OL[i][k] X[k][j] */
            if (!t->Lm) { for (size_t e = 0; e < (size_t)dLo * dRo; e++) out[e] += t->alpha * X[e]; }
            else {
#pragma omp parallel for schedule(static) if (rows_mode && (double)dLo * dLi * dRo > 2e5)
                for (int i = 0; i < dLo; i++)
                    for (int kk = 0; kk < dLi; kk++) {
                        double a = t->alpha * (t->Lt ? t->Lm[(size_t)kk * dLo + i] : t->Lm[(size_t)i * dLi + kk]);
                        for (int j = 0; j < dRo; j++) out[(size_t)i * dRo + j] += a * X[(size_t)kk * dRo + j];
                    }
                flops += 2.0 * dLo * dLi * dRo;
            }
            free(X);
            done++;
        }
    }
    if (flops_out) *flops_out = flops;
    free(start); free(want); free(tasks);
    free_optabs(T, nops, owned, nowned);
    return done;
}


/* The cost measure alone (Table 1 caption: the FLOP count of a GEMM C = A B with shapes
 * (M,K)(K,N) is 2MNK): the same (term, psi block, dot transition) expansion as opair_sigma, no arithmetic.
 * flops_out = sum over tasks of 2 dLi dRi dRo (if the R factor is not the identity) + 2 dLo dLi dRo (if the
 * L factor is not the identity).  values may be NULL (only block presence is used).  Returns the task count. */
int64_t opair_count(const int32_t *secL, int nsecL, const int32_t *secR, int nsecR,
    const int64_t *ops, int nops, const int64_t *blocks, const double *values,
    const int64_t *lin_ptr, const int32_t *lin_op, const double *lin_coef,
    const double *site_ops, const int32_t *site_parity, int nsite,
    const double *term_coef, const int32_t *term_idx, int64_t nterms,
    const int64_t *layout, int64_t npsiblk, int64_t psi_size,
    const int32_t *only_out, int n_only, double *flops_out) {
    static const double dummy = 0.0;
    (void)psi_size;
    problem_t P = make_problem(secL, nsecL, secR, nsecR, ops, nops, blocks, values ? values : &dummy, lin_ptr, lin_op, lin_coef,
                               site_ops, site_parity, nsite, term_coef, term_idx, nterms, layout, npsiblk);
    double **owned; int nowned;
    optab_t *T = build_optabs(&P, &owned, &nowned, 0);
    int64_t ntask;
    task_t *tasks = enumerate_tasks(&P, T, &ntask, 0);
    char *want = (char *)malloc(npsiblk);
    memset(want, n_only > 0 ? 0 : 1, npsiblk);
    for (int i = 0; i < n_only; i++) want[only_out[i]] = 1;
    double flops = 0.0; int64_t done = 0;
    for (int64_t k = 0; k < ntask; k++) {
        const task_t *t = &tasks[k];
        if (!want[t->out_blk]) continue;
        if (t->Rm) flops += 2.0 * t->dLi * t->dRi * t->dRo;
        if (t->Lm) flops += 2.0 * t->dLo * t->dLi * t->dRo;
        done++;
    }
    if (flops_out) *flops_out = flops;
    free(want); free(tasks);
    free_optabs(T, nops, owned, nowned);
    return done;
}

/* Diagonal of H in the psi layout: terms whose four factors are all block-diagonal. */
int64_t opair_hdiag(const int32_t *secL, int nsecL, const int32_t *secR, int nsecR,
    const int64_t *ops, int nops, const int64_t *blocks, const double *values,
    const int64_t *lin_ptr, const int32_t *lin_op, const double *lin_coef,
    const double *site_ops, const int32_t *site_parity, int nsite,
    const double *term_coef, const int32_t *term_idx, int64_t nterms,
    const int64_t *layout, int64_t npsiblk, int64_t psi_size, double *diag) {
    problem_t P = make_problem(secL, nsecL, secR, nsecR, ops, nops, blocks, values, lin_ptr, lin_op, lin_coef,
                               site_ops, site_parity, nsite, term_coef, term_idx, nterms, layout, npsiblk);
    double **owned; int nowned;
    optab_t *T = build_optabs(&P, &owned, &nowned, 1);
    int64_t ntask;
    task_t *tasks = enumerate_tasks(&P, T, &ntask, 1);
    memset(diag, 0, psi_size * sizeof(double));
    for (int64_t k = 0; k < ntask; k++) {
        const task_t *t = &tasks[k];
        double *out = diag + layout[7 * t->out_blk + 6];
        int dL = t->dLi, dR = t->dRi;
        for (int i = 0; i < dL; i++) {
            double l = t->Lm ? t->Lm[(size_t)i * dL + i] : 1.0;
            for (int j = 0; j < dR; j++) {
                double r = t->Rm ? t->Rm[(size_t)j * dR + j] : 1.0;
                out[(size_t)i * dR + j] += t->alpha * l * r;
            }
        }
    }
    free(tasks);
    free_optabs(T, nops, owned, nowned);
    return ntask;
}

/* ------------------------------------------------------------------ O-def: Slater-Condon FCI */
/* Determinants are bit strings over n spin orbitals, bit P set = a+_P present, creation
 * operators in ascending P order (conventions of DESIGN.md).  hso[n*n], V[n^4] = <PQ||RS>. */
static inline int popc(uint64_t x) { return __builtin_popcountll(x); }
static inline int below(uint64_t d, int P) { return popc(d & ((1ULL << P) - 1)); }

/* apply a_P (ann) or a+_P (cre) to bit string with sign; returns 0 if annihilated */
static int apply_ann(uint64_t *d, int P, int *sgn) {
    if (!((*d >> P) & 1)) return 0;
    if (below(*d, P) & 1) *sgn = -*sgn;
    *d &= ~(1ULL << P);
    return 1;
}
static int apply_cre(uint64_t *d, int P, int *sgn) {
    if ((*d >> P) & 1) return 0;
    if (below(*d, P) & 1) *sgn = -*sgn;
    *d |= (1ULL << P);
    return 1;
}

double fci_element(uint64_t bra, uint64_t ket, int n, const double *hso, const double *V) {
#define VV(p, q, r, s) V[(((size_t)(p) * n + (q)) * n + (r)) * n + (s)]
    uint64_t diff = bra ^ ket;
    int nd = popc(diff);
    if (nd == 0) {
        double e = 0.0;
        for (int i = 0; i < n; i++) if ((ket >> i) & 1) {
            e += hso[i * n + i];
            for (int j = 0; j < n; j++) if ((ket >> j) & 1) e += 0.5 * VV(i, j, i, j);
        }
        return e;
    }
    if (nd == 2) {
        int i = __builtin_ctzll(ket & diff), a = __builtin_ctzll(bra & diff);
        int lo = i < a ? i : a, hi = i < a ? a : i;
        uint64_t between = ket & (((1ULL << hi) - 1) & ~((1ULL << (lo + 1)) - 1));
        double ph = (popc(between) & 1) ? -1.0 : 1.0;
        double e = hso[a * n + i];
        for (int j = 0; j < n; j++) if ((ket >> j) & 1) e += VV(a, j, i, j);
        return ph * e;
    }
    if (nd == 4) {
        uint64_t from = ket & diff, to = bra & diff;
        int i = __builtin_ctzll(from), j = 63 - __builtin_clzll(from);
        int a = __builtin_ctzll(to), b = 63 - __builtin_clzll(to);
        uint64_t d = ket; int sgn = 1;
        apply_ann(&d, i, &sgn); apply_ann(&d, j, &sgn); apply_cre(&d, b, &sgn); apply_cre(&d, a, &sgn);
        return sgn * VV(a, b, i, j);
    }
    return 0.0;
#undef VV
}

void fci_dense_h(const uint64_t *dets, int64_t ndet, int n, const double *hso, const double *V, double *H) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < ndet; i++)
        for (int64_t j = 0; j < ndet; j++)
            H[i * ndet + j] = fci_element(dets[i], dets[j], n, hso, V);
}
