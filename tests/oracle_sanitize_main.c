/* Driver for tests/test_oracle_sanitized.py: every entry of the CPU oracle once, on a small jittered grid, built with
 * -fsanitize=address,undefined (sanitizers for the oracle).  Test infrastructure only.
 * Exit code 0 = every call returned what it should; the sanitizers abort the process on a finding. */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

typedef struct orc_mesh orc_mesh;
orc_mesh *orc_build(const double *, int, int64_t, const int32_t *, int64_t, const double *, int *);
void orc_free(orc_mesh *);
int64_t orc_nv(const orc_mesh *);
int64_t orc_nnz(const orc_mesh *);
void orc_get_csr(const orc_mesh *, int64_t *, int32_t *, double *);
void orc_get_area(const orc_mesh *, double *);
void orc_apply_S(const orc_mesh *, const double *, double *);
void orc_apply(const orc_mesh *, double, int, double, const double *, double *, double *);
int orc_solve(const orc_mesh *, const double *, double, int, double, double, int64_t, double *, int64_t *, double *, double *);
double orc_energy(const orc_mesh *, const double *);
void orc_spectrum(const double *, const double *, int, double *, double *);
int orc_dense_solve(const orc_mesh *, const double *, double, int, double, double *);
int orc_build_vector(orc_mesh *, const double *, int, const int32_t *, int64_t, const double *, double);
void orc_get_vector_csr(const orc_mesh *, double *, double *);
void orc_apply_vector(const orc_mesh *, double, int, double, const double *, const double *, double *, double *, double *);
int orc_solve_vector(const orc_mesh *, const double *, const double *, double, int, double, double, int64_t, double *,
                     double *, int64_t *, double *, double *);

static uint64_t state = 88172645463325252ull;
static double rnd(void) {   /* xorshift: uniform in [-1, 1) */
    state ^= state << 13; state ^= state >> 7; state ^= state << 17;
    return (double)(state >> 11) / 4503599627370496.0 - 1.0;
}

#define CHECK(cond) do { if (!(cond)) { fprintf(stderr, "check failed: %s (line %d)\n", #cond, __LINE__); return 1; } } while (0)

static int run(int n, int periodic, int dim) {
    const int n1 = periodic ? n : n + 1;
    const int64_t nv = (int64_t)n1 * n1, nt = 2 * (int64_t)n * n;
    double *coords = malloc((size_t)nv * dim * sizeof(double));
    int32_t *tri = malloc((size_t)nt * 3 * sizeof(int32_t));
    double period[3] = {(double)n, (double)n, 0.0};
    for (int iy = 0; iy < n1; ++iy)
        for (int ix = 0; ix < n1; ++ix) {
            const int64_t v = (int64_t)iy * n1 + ix;
            const double x = ix + 0.2 * rnd(), y = iy + 0.2 * rnd();
            if (dim == 2) { coords[2 * v] = x; coords[2 * v + 1] = y; }
            else {   /* a patch of the unit sphere around latitude 30 degrees: lon, lat from the grid */
                const double lon = 0.02 * x, lat = 0.5 + 0.02 * y;
                coords[3 * v] = cos(lat) * cos(lon); coords[3 * v + 1] = cos(lat) * sin(lon); coords[3 * v + 2] = sin(lat);
            }
        }
    int64_t t = 0;
    for (int cy = 0; cy < n; ++cy)
        for (int cx = 0; cx < n; ++cx) {
            const int x1 = periodic ? (cx + 1) % n : cx + 1, y1 = periodic ? (cy + 1) % n : cy + 1;
            const int32_t v00 = cy * n1 + cx, v10 = cy * n1 + x1, v01 = y1 * n1 + cx, v11 = y1 * n1 + x1;
            if (rnd() > 0.0) { tri[3*t] = v00; tri[3*t+1] = v10; tri[3*t+2] = v11; ++t; tri[3*t] = v00; tri[3*t+1] = v11; tri[3*t+2] = v01; ++t; }
            else             { tri[3*t] = v00; tri[3*t+1] = v10; tri[3*t+2] = v01; ++t; tri[3*t] = v10; tri[3*t+1] = v11; tri[3*t+2] = v01; ++t; }
        }
    int err = 0;
    orc_mesh *m = orc_build(coords, dim, nv, tri, nt, (periodic && dim == 2) ? period : NULL, &err);
    CHECK(m && err == 0 && orc_nv(m) == nv);
    const int64_t nnz = orc_nnz(m);
    int64_t *rp = malloc((size_t)(nv + 1) * sizeof(int64_t));
    int32_t *col = malloc((size_t)nnz * sizeof(int32_t));
    double *val = malloc((size_t)nnz * sizeof(double)), *area = malloc((size_t)nv * sizeof(double));
    orc_get_csr(m, rp, col, val);
    orc_get_area(m, area);
    CHECK(rp[nv] == nnz);
    double *phi = malloc((size_t)nv * sizeof(double)), *psi = malloc((size_t)nv * sizeof(double));
    double *x = malloc((size_t)nv * sizeof(double)), *y = malloc((size_t)nv * sizeof(double));
    double *tmp = malloc((size_t)4 * nv * sizeof(double));
    for (int64_t v = 0; v < nv; ++v) { phi[v] = rnd(); psi[v] = rnd(); }
    orc_apply_S(m, phi, y);
    double e[4], ells[4] = {0.7, 1.5, 3.0, 6.0}, kmid[3], E[3];
    for (int order = 1; order <= 4; ++order) {
        orc_apply(m, 1.3, order, 0.5, phi, y, tmp);
        int64_t it = 0;
        double rec = 0, tru = 0;
        const int st = orc_solve(m, phi, order <= 2 ? 2.0 : 1.2, order, 0.5, 1e-13, 100000, x, &it, &rec, &tru);
        CHECK(st == 0 && rec <= 1e-13 && it > 0);
        if (nv <= 200) CHECK(orc_dense_solve(m, phi, 1.5, order, 0.5, y) == 0);
    }
    for (int j = 0; j < 4; ++j) {
        int64_t it; double rec, tru;
        CHECK(orc_solve(m, phi, ells[j], 1, 0.5, 1e-13, 100000, x, &it, &rec, &tru) == 0);
        e[j] = orc_energy(m, x);
    }
    orc_spectrum(ells, e, 4, kmid, E);
    CHECK(E[0] > 0 && E[1] > 0 && E[2] > 0);
    CHECK(orc_build_vector(m, coords, dim, tri, nt, (periodic && dim == 2) ? period : NULL, dim == 3 ? 1.0 : 0.0) == 0);
    double *dv = malloc((size_t)nnz * sizeof(double)), *tv = malloc((size_t)nnz * sizeof(double));
    orc_get_vector_csr(m, dv, tv);
    for (int order = 1; order <= 2; ++order) {
        int64_t it; double rec, tru;
        orc_apply_vector(m, 1.3, order, 0.5, phi, psi, x, y, tmp);
        CHECK(orc_solve_vector(m, phi, psi, 2.0, order, 0.5, 1e-13, 100000, x, y, &it, &rec, &tru) == 0);
    }
    /* error paths free what they allocated */
    tri[0] = (int32_t)nv + 5;
    CHECK(orc_build(coords, dim, nv, tri, nt, NULL, &err) == NULL && err == 1);
    free(dv); free(tv); free(phi); free(psi); free(x); free(y); free(tmp); free(rp); free(col); free(val); free(area);
    orc_free(m);
    free(coords); free(tri);
    return 0;
}

int main(void) {
    if (run(12, 1, 2)) return 1;     /* periodic planar */
    if (run(9, 0, 2)) return 1;      /* planar with a boundary, 100 vertices: dense path included */
    if (run(10, 0, 3)) return 1;     /* a patch of the sphere: metric terms */
    printf("oracle sanitized run ok\n");
    return 0;
}
