/*
 * ORACLE -- test infrastructure, not product code.
 *
 * A plain, slow, fp64 CPU statement of what the hot path of arXiv 2404.07398 computes, written
 * from the paper (citations "PAPER.md:NN" = /root/reference/PAPER.md line NN) with the readings
 * listed in DESIGN.md.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  It shares no code with paper_2404_07398_b200/ (the CUDA
 * library) and must never be used as a fallback for it.
 *
 * What is computed (notation of BASELINE.json: S = P1 stiffness, M = diag(A_v) lumped mass):
 *   geometry   PAPER.md:57-61   S_vv' = integral grad N_v . grad N_v' dS  (closed form: -1/2 cot of the
 *                               angle opposite edge vv', summed over the triangles sharing the edge);
 *                               boundary term dropped = no-normal-flux condition
 *   mass       PAPER.md:61      M^L = diag(A_v), A_v = median-dual area = sum of area_t/3 (Fig. 1a, :41)
 *   operator   PAPER.md:61,:63  A_l = M + gamma l^2 S           (n = 1)
 *                               A_l = M + gamma l^4 S M^-1 S    (n = 2)      gamma = 1/2
 *                               A_l = M + gamma l^(2n) S (M^-1 S)^(n-1)  (n = 3, 4: "This procedure can be generalized
 *                               to higher-order filters"; the four-Laplacian filter of PAPER.md:201-205)
 *   solve      PAPER.md:113     conjugate gradients on A_l x = M phi started from x0 = phi (the
 *                               Guedot subtraction), Jacobi preconditioner (reading A8),
 *                               stop at ||r||_2 <= tol ||M phi||_2 (reading A6; tol 1e-13 by default)
 *   energy     PAPER.md:31      e_l = 1/2 sum_v A_v x_v^2 / sum_v A_v   ("second moment")
 *   spectrum   PAPER.md:31,:209 k_l = 1/l ; E_j = (e_j - e_j+1)/(k_j - k_j+1) at sqrt(k_j k_j+1) (reading A4)
 *   dense      BASELINE.json    Cholesky solve of the dense A_l for small meshes (cross-check of CG)
 *
 * Pins (tests/test_oracle_pins.py): P1-gradient definition of S by quadrature-free element matrices,
 * 5-point stencil on the uniform grid, equilateral lattice, plane-wave closed form,
 * dense solve, mean conservation, energy monotonicity, icosphere eigenvalues l(l+1).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int64_t nv;       /* vertices */
    int64_t nnz;      /* stored entries of S, diagonal included */
    int64_t *rowptr;  /* [nv+1] */
    int32_t *col;     /* [nnz] ascending within a row */
    double *val;      /* [nnz] */
    double *area;     /* [nv] A_v */
    double *gdiag;    /* [nv] diag(S M^-1 S)_v = sum_j S_vj^2 / A_j */
    double *sdiag;    /* [nv] S_vv */
    /* vector filter (orc_build_vector), on the sparsity pattern of S: */
    double *dval;     /* [nnz] D~_vv'/l^2 = int (grad N_v . grad N_v' + (R_e^-2 + m^2) N_v N_v') dS            */
    double *tval;     /* [nnz] T_vv'/l^2  = int m (-N_v' dx N_v + N_v dx N_v') dS   (antisymmetric, zero diagonal) */
} orc_mesh;

static void edge_vec(const double *coords, int dim, const double *period, int64_t from, int64_t to,
                     double e[3]) {
    /* e = x_to - x_from, minimum image on periodic axes: d -= P round(d/P) */
    e[0] = e[1] = e[2] = 0.0;
    for (int d = 0; d < dim; ++d) {
        double v = coords[to * dim + d] - coords[from * dim + d];
        if (period && period[d] > 0.0) v -= period[d] * nearbyint(v / period[d]);
        e[d] = v;
    }
}

void orc_free(orc_mesh *m) {
    if (!m) return;
    free(m->rowptr); free(m->col); free(m->val); free(m->area); free(m->gdiag); free(m->sdiag);
    free(m->dval); free(m->tval);
    free(m);
}

/* Build S (CSR) and A_v.  Returns NULL and sets *err: 1 bad index, 2 degenerate triangle,
 * 3 vertex in no triangle (A_v = 0), 4 out of memory. */
orc_mesh *orc_build(const double *coords, int dim, int64_t nv, const int32_t *tri, int64_t nt,
                    const double *period, int *err) {
    *err = 0;
    orc_mesh *m = (orc_mesh *)calloc(1, sizeof(orc_mesh));
    int64_t *cap = (int64_t *)calloc((size_t)nv + 1, sizeof(int64_t));
    if (!m || !cap) { *err = 4; free(cap); orc_free(m); return NULL; }
    m->nv = nv;
    /* capacity: every triangle adds two off-diagonal contributions to each of its three rows */
    for (int64_t t = 0; t < nt; ++t)
        for (int c = 0; c < 3; ++c) {
            int64_t v = tri[3 * t + c];
            if (v < 0 || v >= nv) { *err = 1; free(cap); orc_free(m); return NULL; }
            cap[v + 1] += 2;
        }
    for (int64_t t = 0; t < nt; ++t)
        if (tri[3 * t] == tri[3 * t + 1] || tri[3 * t] == tri[3 * t + 2] || tri[3 * t + 1] == tri[3 * t + 2]) {
            *err = 1; free(cap); orc_free(m); return NULL;
        }
    for (int64_t v = 0; v < nv; ++v) cap[v + 1] += cap[v] + 1; /* +1: the diagonal */
    int64_t total = cap[nv];
    int32_t *tc = (int32_t *)malloc((size_t)total * sizeof(int32_t));
    double *tv = (double *)malloc((size_t)total * sizeof(double));
    int64_t *fill = (int64_t *)calloc((size_t)nv, sizeof(int64_t));
    m->area = (double *)calloc((size_t)nv, sizeof(double));
    if (!tc || !tv || !fill || !m->area) { *err = 4; goto fail; }

    for (int64_t t = 0; t < nt; ++t) {
        double tarea = 0.0;
        for (int c = 0; c < 3; ++c) {
            /* corner c, the other two vertices a, b: the angle at c is opposite edge ab */
            int64_t vc = tri[3 * t + c], va = tri[3 * t + (c + 1) % 3], vb = tri[3 * t + (c + 2) % 3];
            double e1[3], e2[3];
            edge_vec(coords, dim, period, vc, va, e1);
            edge_vec(coords, dim, period, vc, vb, e2);
            double cx = e1[1] * e2[2] - e1[2] * e2[1];
            double cy = e1[2] * e2[0] - e1[0] * e2[2];
            double cz = e1[0] * e2[1] - e1[1] * e2[0];
            double cr = sqrt(cx * cx + cy * cy + cz * cz);          /* = 2 * area, unsigned */
            double dot = e1[0] * e2[0] + e1[1] * e2[1] + e1[2] * e2[2];
            double n1 = e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2];
            double n2 = e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2];
            if (!(cr > 1e-14 * (n1 + n2))) { *err = 2; goto fail; }
            double w = -0.5 * dot / cr;                              /* -1/2 cot(angle at c) */
            tc[cap[va] + fill[va]] = (int32_t)vb; tv[cap[va] + fill[va]] = w; fill[va]++;
            tc[cap[vb] + fill[vb]] = (int32_t)va; tv[cap[vb] + fill[vb]] = w; fill[vb]++;
            if (c == 0) tarea = 0.5 * cr;
        }
        for (int c = 0; c < 3; ++c) m->area[tri[3 * t + c]] += tarea / 3.0;
    }
    for (int64_t v = 0; v < nv; ++v)
        if (!(m->area[v] > 0.0)) { *err = 3; goto fail; }

    /* per row: sort by column, merge duplicates, add the diagonal S_vv = -sum of off-diagonals */
    m->rowptr = (int64_t *)calloc((size_t)nv + 1, sizeof(int64_t));
    if (!m->rowptr) { *err = 4; goto fail; }
    for (int64_t v = 0; v < nv; ++v) {
        int64_t b = cap[v], n = fill[v];
        for (int64_t i = 1; i < n; ++i) {          /* insertion sort, stable */
            int32_t c = tc[b + i]; double x = tv[b + i]; int64_t j = i;
            while (j > 0 && tc[b + j - 1] > c) { tc[b + j] = tc[b + j - 1]; tv[b + j] = tv[b + j - 1]; --j; }
            tc[b + j] = c; tv[b + j] = x;
        }
        int64_t u = 0;
        for (int64_t i = 0; i < n; ++i) {
            if (u > 0 && tc[b + u - 1] == tc[b + i]) tv[b + u - 1] += tv[b + i];
            else { tc[b + u] = tc[b + i]; tv[b + u] = tv[b + i]; ++u; }
        }
        fill[v] = u;
        m->rowptr[v + 1] = m->rowptr[v] + u + 1;
    }
    m->nnz = m->rowptr[nv];
    m->col = (int32_t *)malloc((size_t)m->nnz * sizeof(int32_t));
    m->val = (double *)malloc((size_t)m->nnz * sizeof(double));
    m->sdiag = (double *)malloc((size_t)nv * sizeof(double));
    m->gdiag = (double *)malloc((size_t)nv * sizeof(double));
    if (!m->col || !m->val || !m->sdiag || !m->gdiag) { *err = 4; goto fail; }
    for (int64_t v = 0; v < nv; ++v) {
        int64_t b = cap[v], n = fill[v], o = m->rowptr[v];
        double diag = 0.0;
        for (int64_t i = 0; i < n; ++i) diag -= tv[b + i];
        int placed = 0;
        for (int64_t i = 0; i < n; ++i) {
            if (!placed && tc[b + i] > v) { m->col[o] = (int32_t)v; m->val[o] = diag; ++o; placed = 1; }
            m->col[o] = tc[b + i]; m->val[o] = tv[b + i]; ++o;
        }
        if (!placed) { m->col[o] = (int32_t)v; m->val[o] = diag; ++o; }
        m->sdiag[v] = diag;
    }
    for (int64_t v = 0; v < nv; ++v) {
        double g = 0.0;
        for (int64_t i = m->rowptr[v]; i < m->rowptr[v + 1]; ++i)
            g += m->val[i] * m->val[i] / m->area[m->col[i]];
        m->gdiag[v] = g;
    }
    free(tc); free(tv); free(fill); free(cap);
    return m;
fail:
    free(tc); free(tv); free(fill); free(cap); orc_free(m);
    return NULL;
}

int64_t orc_nv(const orc_mesh *m) { return m->nv; }
int64_t orc_nnz(const orc_mesh *m) { return m->nnz; }
void orc_get_csr(const orc_mesh *m, int64_t *rowptr, int32_t *col, double *val) {
    memcpy(rowptr, m->rowptr, (size_t)(m->nv + 1) * sizeof(int64_t));
    memcpy(col, m->col, (size_t)m->nnz * sizeof(int32_t));
    memcpy(val, m->val, (size_t)m->nnz * sizeof(double));
}
void orc_get_area(const orc_mesh *m, double *area) { memcpy(area, m->area, (size_t)m->nv * sizeof(double)); }

/* y = S p */
void orc_apply_S(const orc_mesh *m, const double *p, double *y) {
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < m->nv; ++v) {
        double s = 0.0;
        for (int64_t i = m->rowptr[v]; i < m->rowptr[v + 1]; ++i) s += m->val[i] * p[m->col[i]];
        y[v] = s;
    }
}

/* out = A_l p,  A_l = M + gamma l^(2n) S (M^-1 S)^(n-1)   (PAPER.md:61 n=1, PAPER.md:63 n=2 and "higher-order").
 * tmp: scratch [nv], used for n >= 2 only. */
void orc_apply(const orc_mesh *m, double ell, int n, double gamma, const double *p, double *out, double *tmp) {
    const double c = gamma * pow(ell, 2.0 * n);
    if (n > 2) {
        /* the two-step derivation of PAPER.md:63 repeated: psi_1 = M^-1 S p, psi_k = M^-1 S psi_k-1, out = M p + c S psi_n-1 */
        double *psi = (double *)malloc((size_t)m->nv * sizeof(double));
        orc_apply_S(m, p, tmp);
        for (int64_t v = 0; v < m->nv; ++v) psi[v] = tmp[v] / m->area[v];
        for (int k = 2; k < n; ++k) {
            orc_apply_S(m, psi, tmp);
            for (int64_t v = 0; v < m->nv; ++v) psi[v] = tmp[v] / m->area[v];
        }
        orc_apply_S(m, psi, out);
        for (int64_t v = 0; v < m->nv; ++v) out[v] = m->area[v] * p[v] + c * out[v];
        free(psi);
        return;
    }
    if (n == 1) {
        orc_apply_S(m, p, out);
#pragma omp parallel for schedule(static)
        for (int64_t v = 0; v < m->nv; ++v) out[v] = m->area[v] * p[v] + c * out[v];
    } else {
        orc_apply_S(m, p, tmp);                                   /* M psi = S p */
#pragma omp parallel for schedule(static)
        for (int64_t v = 0; v < m->nv; ++v) tmp[v] /= m->area[v];
        orc_apply_S(m, tmp, out);
#pragma omp parallel for schedule(static)
        for (int64_t v = 0; v < m->nv; ++v) out[v] = m->area[v] * p[v] + c * out[v];
    }
}

/* diag(S (M^-1 S)^(n-1))_v for n >= 3, exactly: column v of the operator is built as a sparse vector, one factor at a
 * time (u <- S u, u <- u / A), and its entry v is read off.  Plain and slow: a dense scratch vector with a list of the
 * touched entries, O(ring size) per factor. */
static double diag_higher(const orc_mesh *m, int64_t v, int n, double *u, double *w, int64_t *tu, int64_t *tw, char *mark) {
    int64_t nu = 1;
    u[v] = 1.0; tu[0] = v;
    double result = 0.0;
    for (int k = 0; k < n; ++k) {
        /* w = S u */
        int64_t nw = 0;
        for (int64_t a = 0; a < nu; ++a) {
            int64_t j = tu[a];
            for (int64_t i = m->rowptr[j]; i < m->rowptr[j + 1]; ++i) {       /* S symmetric: column j = row j */
                int64_t r = m->col[i];
                if (!mark[r]) { mark[r] = 1; w[r] = 0.0; tw[nw++] = r; }
                w[r] += m->val[i] * u[j];
            }
        }
        for (int64_t a = 0; a < nu; ++a) u[tu[a]] = 0.0;
        if (k == n - 1) result = mark[v] ? w[v] : 0.0;
        /* u = M^-1 w */
        for (int64_t a = 0; a < nw; ++a) { int64_t r = tw[a]; u[r] = w[r] / m->area[r]; tu[a] = r; mark[r] = 0; }
        nu = nw;
    }
    for (int64_t a = 0; a < nu; ++a) u[tu[a]] = 0.0;
    return result;
}

static double dot(int64_t n, const double *a, const double *b) {
    double s = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : s)
    for (int64_t i = 0; i < n; ++i) s += a[i] * b[i];
    return s;
}

/* Jacobi-preconditioned CG on A_l x = M phi from x0 = phi.
 * Stops when the recursive residual satisfies ||r||_2 <= tol ||M phi||_2, or at max_iter.
 * Outputs: x [nv]; *iters; *rec_res = ||r||/||M phi|| (recursive); *true_res = ||M phi - A_l x||/||M phi||.
 * Returns 0 converged, 1 iteration cap, 2 breakdown (p.Ap <= 0 or non-finite), 4 out of memory. */
int orc_solve(const orc_mesh *m, const double *phi, double ell, int n, double gamma, double tol,
              int64_t max_iter, double *x, int64_t *iters, double *rec_res, double *true_res) {
    const int64_t nv = m->nv;
    const double c = gamma * pow(ell, 2.0 * n);
    double *b = (double *)malloc((size_t)nv * sizeof(double));
    double *r = (double *)malloc((size_t)nv * sizeof(double));
    double *z = (double *)malloc((size_t)nv * sizeof(double));
    double *p = (double *)malloc((size_t)nv * sizeof(double));
    double *q = (double *)malloc((size_t)nv * sizeof(double));
    double *d = (double *)malloc((size_t)nv * sizeof(double));
    double *tmp = (double *)malloc((size_t)nv * sizeof(double));
    int status = 1;
    if (!b || !r || !z || !p || !q || !d || !tmp) { status = 4; goto done; }
    for (int64_t v = 0; v < nv; ++v) {
        b[v] = m->area[v] * phi[v];
        x[v] = phi[v];
        d[v] = m->area[v] + c * (n == 1 ? m->sdiag[v] : m->gdiag[v]);   /* diag(A_l) */
    }
    if (n > 2) {   /* diag(A_l) for the higher orders, computed exactly row by row */
        double *u = (double *)calloc((size_t)nv, sizeof(double)), *w = (double *)calloc((size_t)nv, sizeof(double));
        int64_t *tu = (int64_t *)malloc((size_t)nv * sizeof(int64_t)), *tw = (int64_t *)malloc((size_t)nv * sizeof(int64_t));
        char *mark = (char *)calloc((size_t)nv, 1);
        if (!u || !w || !tu || !tw || !mark) { free(u); free(w); free(tu); free(tw); free(mark); status = 4; goto done; }
        for (int64_t v = 0; v < nv; ++v) d[v] = m->area[v] + c * diag_higher(m, v, n, u, w, tu, tw, mark);
        free(u); free(w); free(tu); free(tw); free(mark);
    }
    orc_apply(m, ell, n, gamma, x, q, tmp);
    for (int64_t v = 0; v < nv; ++v) { r[v] = b[v] - q[v]; z[v] = r[v] / d[v]; p[v] = z[v]; }
    double bb = dot(nv, b, b);
    double rho = dot(nv, r, z);
    double rr = dot(nv, r, r);
    int64_t it = 0;
    if (rr <= tol * tol * bb) status = 0;
    while (status == 1 && it < max_iter) {
        orc_apply(m, ell, n, gamma, p, q, tmp);
        double pq = dot(nv, p, q);
        if (!(pq > 0.0) || !isfinite(pq)) { status = 2; break; }
        double alpha = rho / pq;
#pragma omp parallel for schedule(static)
        for (int64_t v = 0; v < nv; ++v) { x[v] += alpha * p[v]; r[v] -= alpha * q[v]; z[v] = r[v] / d[v]; }
        double rho_new = dot(nv, r, z);
        rr = dot(nv, r, r);
        ++it;
        if (rr <= tol * tol * bb) { status = 0; break; }
        double beta = rho_new / rho;
        rho = rho_new;
#pragma omp parallel for schedule(static)
        for (int64_t v = 0; v < nv; ++v) p[v] = z[v] + beta * p[v];
    }
    *iters = it;
    *rec_res = bb > 0.0 ? sqrt(rr / bb) : 0.0;
    orc_apply(m, ell, n, gamma, x, q, tmp);
    for (int64_t v = 0; v < nv; ++v) q[v] = b[v] - q[v];
    *true_res = bb > 0.0 ? sqrt(dot(nv, q, q) / bb) : 0.0;
done:
    free(b); free(r); free(z); free(p); free(q); free(d); free(tmp);
    return status;
}

/* e = 1/2 sum_v A_v x_v^2 / sum_v A_v  ("second moment"; reading A4) */
double orc_energy(const orc_mesh *m, const double *x) {
    double s = 0.0, a = 0.0;
    for (int64_t v = 0; v < m->nv; ++v) { s += m->area[v] * x[v] * x[v]; a += m->area[v]; }
    return 0.5 * s / a;
}

/* k_j = 1/l_j; E_j = (e_j - e_j+1)/(k_j - k_j+1), k_mid_j = sqrt(k_j k_j+1), j < L-1 */
void orc_spectrum(const double *ells, const double *e, int L, double *k_mid, double *E) {
    for (int j = 0; j + 1 < L; ++j) {
        double k0 = 1.0 / ells[j], k1 = 1.0 / ells[j + 1];
        E[j] = (e[j] - e[j + 1]) / (k0 - k1);
        k_mid[j] = sqrt(k0 * k1);
    }
}

/* Dense check path: build A_l densely, Cholesky-factorise, solve A_l x = M phi.  O(nv^3): small meshes only.
 * Returns 0 ok, 2 not positive definite, 4 out of memory. */
int orc_dense_solve(const orc_mesh *m, const double *phi, double ell, int n, double gamma, double *x) {
    const int64_t nv = m->nv;
    const double c = gamma * pow(ell, 2.0 * n);
    double *Sd = (double *)calloc((size_t)(nv * nv), sizeof(double));
    double *A = (double *)calloc((size_t)(nv * nv), sizeof(double));
    if (!Sd || !A) { free(Sd); free(A); return 4; }
    for (int64_t v = 0; v < nv; ++v)
        for (int64_t i = m->rowptr[v]; i < m->rowptr[v + 1]; ++i) Sd[v * nv + m->col[i]] = m->val[i];
    if (n == 1) {
        for (int64_t i = 0; i < nv * nv; ++i) A[i] = c * Sd[i];
    } else if (n == 2) {
        for (int64_t i = 0; i < nv; ++i)
            for (int64_t k = 0; k < nv; ++k) {
                double sik = Sd[i * nv + k];
                if (sik == 0.0) continue;
                double f = c * sik / m->area[k];
                for (int64_t j = 0; j < nv; ++j) A[i * nv + j] += f * Sd[k * nv + j];
            }
    } else {
        /* A = c S (M^-1 S)^(n-1): P <- S, then n-1 times P <- P M^-1 S */
        double *P = (double *)malloc((size_t)(nv * nv) * sizeof(double));
        double *Q = (double *)calloc((size_t)(nv * nv), sizeof(double));
        if (!P || !Q) { free(P); free(Q); free(Sd); free(A); return 4; }
        memcpy(P, Sd, (size_t)(nv * nv) * sizeof(double));
        for (int f = 1; f < n; ++f) {
            memset(Q, 0, (size_t)(nv * nv) * sizeof(double));
            for (int64_t i = 0; i < nv; ++i)
                for (int64_t k = 0; k < nv; ++k) {
                    double pik = P[i * nv + k];
                    if (pik == 0.0) continue;
                    double g = pik / m->area[k];
                    for (int64_t j = 0; j < nv; ++j) Q[i * nv + j] += g * Sd[k * nv + j];
                }
            double *T = P; P = Q; Q = T;
        }
        for (int64_t i = 0; i < nv * nv; ++i) A[i] = c * P[i];
        free(P); free(Q);
    }
    for (int64_t v = 0; v < nv; ++v) A[v * nv + v] += m->area[v];
    /* Cholesky A = L L^T, lower triangle in place */
    for (int64_t j = 0; j < nv; ++j) {
        double s = A[j * nv + j];
        for (int64_t k = 0; k < j; ++k) s -= A[j * nv + k] * A[j * nv + k];
        if (!(s > 0.0)) { free(Sd); free(A); return 2; }
        double ljj = sqrt(s);
        A[j * nv + j] = ljj;
        for (int64_t i = j + 1; i < nv; ++i) {
            double t = A[i * nv + j];
            for (int64_t k = 0; k < j; ++k) t -= A[i * nv + k] * A[j * nv + k];
            A[i * nv + j] = t / ljj;
        }
    }
    for (int64_t i = 0; i < nv; ++i) {              /* L y = M phi */
        double t = m->area[i] * phi[i];
        for (int64_t k = 0; k < i; ++k) t -= A[i * nv + k] * x[k];
        x[i] = t / A[i * nv + i];
    }
    for (int64_t i = nv - 1; i >= 0; --i) {         /* L^T x = y */
        double t = x[i];
        for (int64_t k = i + 1; k < nv; ++k) t -= A[k * nv + i] * x[k];
        x[i] = t / A[i * nv + i];
    }
    free(Sd); free(A);
    return 0;
}

int orc_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}


/* ------------------------------------------------------------------------------------------------------------------
 * Vector filter with metric terms (section 2.1.2): the coarse-grained velocity (u, v) = (zonal,
 * meridional) at the vertices of a mesh on the sphere solves the 2V x 2V system
 *     S_2 = M_2 + gamma l^2 D_2            (n = 1),      S_2 = M_2 + gamma l^4 D_2 M_2^-1 D_2     (n = 2),
 *     D_2 = [ D~  T ; -T  D~ ],  M_2 = diag(M, M),  M = diag(A_v)  (lumped, as in the scalar case and as PAPER.md:89
 *     writes for the biharmonic form),
 *     D~_vv' = int (grad N_v . grad N_v' + (R_e^-2 + m^2) N_v N_v') dS,
 *     T_vv'  = int m (-N_v' dx N_v + N_v dx N_v') dS,      m = tan(theta) / R_e "taken constant on triangles".
 * Readings: the triangles are the flat 3-D triangles of the mesh; theta and the zonal unit
 * vector are those of the triangle's centroid; dx N = grad N . e_east; int N_v N_v' = area (1 + delta_vv') / 12 and
 * int N_v = area / 3 (exact P1 integrals).  T is antisymmetric, so D_2 is symmetric; it is the weak form of the
 * vector Laplacian, positive semidefinite.  A planar mesh (dim = 2) has no metric terms: m = 0 and 1/R_e = 0.
 * Returns 0, or 4 out of memory. */
static int64_t find_col(const orc_mesh *m, int64_t row, int64_t c) {
    for (int64_t i = m->rowptr[row]; i < m->rowptr[row + 1]; ++i)
        if (m->col[i] == c) return i;
    return -1;
}

int orc_build_vector(orc_mesh *m, const double *coords, int dim, const int32_t *tri, int64_t nt, const double *period,
                     double radius) {
    free(m->dval); free(m->tval);
    m->dval = (double *)calloc((size_t)m->nnz, sizeof(double));
    m->tval = (double *)calloc((size_t)m->nnz, sizeof(double));
    if (!m->dval || !m->tval) return 4;
    const double inv_r = (dim == 3 && radius > 0.0) ? 1.0 / radius : 0.0;
    for (int64_t t = 0; t < nt; ++t) {
        int64_t v[3] = {tri[3 * t], tri[3 * t + 1], tri[3 * t + 2]};
        double x[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
        for (int d = 0; d < dim; ++d) x[0][d] = coords[v[0] * dim + d];
        for (int c = 1; c < 3; ++c) {                      /* minimum image on periodic axes, as in orc_build */
            double e[3];
            edge_vec(coords, dim, period, v[0], v[c], e);
            for (int d = 0; d < dim; ++d) x[c][d] = x[0][d] + e[d];
        }
        /* unit normal, area, P1 gradients in the triangle's plane: grad N_a = n x (x_c - x_b) / (2 area) */
        double e1[3], e2[3], nrm[3];
        for (int d = 0; d < 3; ++d) { e1[d] = x[1][d] - x[0][d]; e2[d] = x[2][d] - x[0][d]; }
        nrm[0] = e1[1] * e2[2] - e1[2] * e2[1];
        nrm[1] = e1[2] * e2[0] - e1[0] * e2[2];
        nrm[2] = e1[0] * e2[1] - e1[1] * e2[0];
        double cr = sqrt(nrm[0] * nrm[0] + nrm[1] * nrm[1] + nrm[2] * nrm[2]);
        double area = 0.5 * cr;
        for (int d = 0; d < 3; ++d) nrm[d] /= cr;
        double g[3][3];
        for (int a = 0; a < 3; ++a) {
            int b = (a + 1) % 3, c = (a + 2) % 3;
            double ed[3] = {x[c][0] - x[b][0], x[c][1] - x[b][1], x[c][2] - x[b][2]};
            g[a][0] = (nrm[1] * ed[2] - nrm[2] * ed[1]) / cr;
            g[a][1] = (nrm[2] * ed[0] - nrm[0] * ed[2]) / cr;
            g[a][2] = (nrm[0] * ed[1] - nrm[1] * ed[0]) / cr;
        }
        /* metric factor and zonal direction at the centroid */
        double mt = 0.0, east[3] = {1.0, 0.0, 0.0};
        if (dim == 3 && inv_r > 0.0) {
            double cx = (x[0][0] + x[1][0] + x[2][0]) / 3.0, cy = (x[0][1] + x[1][1] + x[2][1]) / 3.0;
            double cz = (x[0][2] + x[1][2] + x[2][2]) / 3.0;
            double rho = sqrt(cx * cx + cy * cy);
            mt = (cz / rho) * inv_r;                       /* tan(theta) / R_e */
            east[0] = -cy / rho; east[1] = cx / rho; east[2] = 0.0;
        }
        double gx[3];
        for (int a = 0; a < 3; ++a) gx[a] = g[a][0] * east[0] + g[a][1] * east[1] + g[a][2] * east[2];
        const double mass_c = inv_r * inv_r + mt * mt;
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                int64_t i = find_col(m, v[a], v[b]);
                double gg = g[a][0] * g[b][0] + g[a][1] * g[b][1] + g[a][2] * g[b][2];
                m->dval[i] += area * gg + mass_c * area * (a == b ? 2.0 : 1.0) / 12.0;
                m->tval[i] += mt * (area / 3.0) * (gx[b] - gx[a]);     /* row v = v[a], column v' = v[b] */
            }
    }
    return 0;
}

void orc_get_vector_csr(const orc_mesh *m, double *dval, double *tval) {
    memcpy(dval, m->dval, (size_t)m->nnz * sizeof(double));
    memcpy(tval, m->tval, (size_t)m->nnz * sizeof(double));
}

/* (yu, yv) = D_2 (pu, pv) / l^2 */
static void apply_D2(const orc_mesh *m, const double *pu, const double *pv, double *yu, double *yv) {
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < m->nv; ++v) {
        double su = 0.0, sv = 0.0;
        for (int64_t i = m->rowptr[v]; i < m->rowptr[v + 1]; ++i) {
            int64_t j = m->col[i];
            su += m->dval[i] * pu[j] + m->tval[i] * pv[j];
            sv += m->dval[i] * pv[j] - m->tval[i] * pu[j];
        }
        yu[v] = su; yv[v] = sv;
    }
}

/* (outu, outv) = S_2 (pu, pv);  tmp: scratch [4 nv] for n = 2 */
void orc_apply_vector(const orc_mesh *m, double ell, int n, double gamma, const double *pu, const double *pv,
                      double *outu, double *outv, double *tmp) {
    const double c = gamma * pow(ell, 2.0 * n);
    const int64_t nv = m->nv;
    if (n == 1) {
        apply_D2(m, pu, pv, outu, outv);
    } else {
        double *tu = tmp, *tv = tmp + nv;
        apply_D2(m, pu, pv, tu, tv);
        for (int64_t v = 0; v < nv; ++v) { tu[v] /= m->area[v]; tv[v] /= m->area[v]; }
        apply_D2(m, tu, tv, outu, outv);
    }
    for (int64_t v = 0; v < nv; ++v) {
        outu[v] = m->area[v] * pu[v] + c * outu[v];
        outv[v] = m->area[v] * pv[v] + c * outv[v];
    }
}

/* Jacobi-preconditioned CG on S_2 (x_u, x_v) = M_2 (u, v) from x0 = (u, v), one residual norm over both
 * components: ||r||_2 <= tol ||M_2 (u, v)||_2.  Same outputs and return codes as orc_solve. */
int orc_solve_vector(const orc_mesh *m, const double *u, const double *v, double ell, int n, double gamma, double tol,
                     int64_t max_iter, double *xu, double *xv, int64_t *iters, double *rec_res, double *true_res) {
    const int64_t nv = m->nv, N = 2 * m->nv;
    const double c = gamma * pow(ell, 2.0 * n);
    double *b = (double *)malloc((size_t)N * sizeof(double)), *r = (double *)malloc((size_t)N * sizeof(double));
    double *z = (double *)malloc((size_t)N * sizeof(double)), *p = (double *)malloc((size_t)N * sizeof(double));
    double *q = (double *)malloc((size_t)N * sizeof(double)), *d = (double *)malloc((size_t)N * sizeof(double));
    double *x = (double *)malloc((size_t)N * sizeof(double)), *tmp = (double *)malloc((size_t)N * sizeof(double));
    int status = 1;
    if (!b || !r || !z || !p || !q || !d || !x || !tmp) { status = 4; goto done; }
    for (int64_t i = 0; i < nv; ++i) {
        /* diag(S_2): n = 1: A_v + c D~_vv;  n = 2: A_v + c sum_j (D~_vj^2 + T_vj^2) / A_j  (D_2 symmetric, T_vv = 0) */
        double dg = 0.0;
        for (int64_t k = m->rowptr[i]; k < m->rowptr[i + 1]; ++k) {
            if (n == 1) { if (m->col[k] == i) dg = m->dval[k]; }
            else dg += (m->dval[k] * m->dval[k] + m->tval[k] * m->tval[k]) / m->area[m->col[k]];
        }
        d[i] = d[nv + i] = m->area[i] + c * dg;
        b[i] = m->area[i] * u[i]; b[nv + i] = m->area[i] * v[i];
        x[i] = u[i]; x[nv + i] = v[i];
    }
    orc_apply_vector(m, ell, n, gamma, x, x + nv, q, q + nv, tmp);
    for (int64_t i = 0; i < N; ++i) { r[i] = b[i] - q[i]; z[i] = r[i] / d[i]; p[i] = z[i]; }
    double bb = dot(N, b, b), rho = dot(N, r, z), rr = dot(N, r, r);
    int64_t it = 0;
    if (rr <= tol * tol * bb) status = 0;
    while (status == 1 && it < max_iter) {
        orc_apply_vector(m, ell, n, gamma, p, p + nv, q, q + nv, tmp);
        double pq = dot(N, p, q);
        if (!(pq > 0.0) || !isfinite(pq)) { status = 2; break; }
        double alpha = rho / pq;
        for (int64_t i = 0; i < N; ++i) { x[i] += alpha * p[i]; r[i] -= alpha * q[i]; z[i] = r[i] / d[i]; }
        double rho_new = dot(N, r, z);
        rr = dot(N, r, r);
        ++it;
        if (rr <= tol * tol * bb) { status = 0; break; }
        double beta = rho_new / rho;
        rho = rho_new;
        for (int64_t i = 0; i < N; ++i) p[i] = z[i] + beta * p[i];
    }
    *iters = it;
    *rec_res = bb > 0.0 ? sqrt(rr / bb) : 0.0;
    orc_apply_vector(m, ell, n, gamma, x, x + nv, q, q + nv, tmp);
    for (int64_t i = 0; i < N; ++i) q[i] = b[i] - q[i];
    *true_res = bb > 0.0 ? sqrt(dot(N, q, q) / bb) : 0.0;
    memcpy(xu, x, (size_t)nv * sizeof(double));
    memcpy(xv, x + nv, (size_t)nv * sizeof(double));
done:
    free(b); free(r); free(z); free(p); free(q); free(d); free(x); free(tmp);
    return status;
}
