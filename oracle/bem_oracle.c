/*
 * bem_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, direct O(N * 3T) CPU evaluation in fp64 of the discretised
 * boundary-element operator  y = S[q] - D[phi]  of arXiv 1905.01341
 * (Eqs. 11-13) at the mesh vertices (collocation at vertices,
 * PAPER.md:152).  It is the oracle the CUDA library is checked against and the
 * `cpu_baseline` that bench.py times.  It shares no code with
 * paper_1905_01341_b200/ and must only be used from tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke().
 *
 * Two quadrature modes (readings R1-R5 in DESIGN.md):
 *   G3  3-point Gauss per flat triangle with P1 (linear) densities, plus the
 *       "high-order minus low-order" correction (ref. [45]) on the
 *       near set N(i); "high order" = the exact flat-triangle integral, obtained
 *       here by adaptive subdivision + Gauss-Legendre (never by the analytic
 *       formulas the CUDA library uses).
 *   V1  the paper's own lumped rule, Eq. 17, with the singular
 *       diagonal from the identities Eqs. 19-21.
 *
 * Sign convention: the normal N points out of the bubble into
 * the liquid;  G = 1/(4 pi |r-r'|),  dG/dn(r') = n(r').(r-r') / (4 pi |r-r'|^3).
 *
 * Pinned by tests/test_oracle_pins.py (sphere eigen-relations, solid-angle
 * identity, closed-form incident weights, brute-force quadrature, V1
 * identities, manufactured exterior fields; the point sums by the mean-value
 * property of the sphere, hand-computed cube corners, Gauss' theorem and a
 * finite difference; the off-surface evaluation by Gauss' theorem and Green's
 * representation of a manufactured exterior field).  No function is unpinned.  Nothing here is tuned for speed:
 * rows are independent and run under `#pragma omp parallel for`, that is all.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define FOUR_PI 12.566370614359172953850573533118

/* ------------------------------------------------------------------ */
/* Gauss-Legendre nodes on [0,1] by Newton iteration on P_n            */
/* ------------------------------------------------------------------ */
static void gauss_legendre01(int n, double *x, double *w)
{
    for (int i = 0; i < n; ++i) {
        double z = cos(M_PI * (i + 0.75) / (n + 0.5));
        double pp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) {
                double p3 = p2;
                p2 = p1;
                p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
            }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        x[i] = 0.5 * (1.0 - z);          /* map [-1,1] -> [0,1], reversed order is irrelevant */
        w[i] = 1.0 / ((1.0 - z * z) * pp * pp);   /* = (2/((1-z^2) pp^2)) / 2 */
    }
}

#define GL_SMALL 8
#define GL_BIG 32
static double gl8_x[GL_SMALL], gl8_w[GL_SMALL];
static double gl32_x[GL_BIG], gl32_w[GL_BIG];
static int gl_ready = 0;

static void gl_init(void)
{
    if (gl_ready) return;
#pragma omp critical(bem_oracle_gl_init)
    {
        if (!gl_ready) {
            gauss_legendre01(GL_SMALL, gl8_x, gl8_w);
            gauss_legendre01(GL_BIG, gl32_x, gl32_w);
            gl_ready = 1;
        }
    }
}

/* ------------------------------------------------------------------ */
/* small vector helpers                                                */
/* ------------------------------------------------------------------ */
static inline void sub3(const double *a, const double *b, double *c)
{ c[0] = a[0] - b[0]; c[1] = a[1] - b[1]; c[2] = a[2] - b[2]; }
static inline double dot3(const double *a, const double *b)
{ return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static inline void cross3(const double *a, const double *b, double *c)
{ c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0]; }

/* Neumaier compensated accumulator: the terms are fp64, only the running sum
 * over millions of triangles is protected against cancellation. */
typedef struct { double s, c; } ksum;
static inline void ksum_add(ksum *k, double v)
{
    double t = k->s + v;
    if (fabs(k->s) >= fabs(v)) k->c += (k->s - t) + v; else k->c += (v - t) + k->s;
    k->s = t;
}
static inline double ksum_get(const ksum *k) { return k->s + k->c; }

/* ------------------------------------------------------------------ */
/* triangle geometry: area, unit normal, 3 Gauss points  */
/* ------------------------------------------------------------------ */
static const double G3_LAMBDA[3][3] = {
    {2.0 / 3.0, 1.0 / 6.0, 1.0 / 6.0},
    {1.0 / 6.0, 2.0 / 3.0, 1.0 / 6.0},
    {1.0 / 6.0, 1.0 / 6.0, 2.0 / 3.0}};

typedef struct {
    double r[3][3];   /* vertices */
    double A;         /* area */
    double N[3];      /* unit normal (e1 x e2)/|e1 x e2| : out of the bubble */
    double y[3][3];   /* Gauss points */
    double c[3];      /* centroid */
    double d2;        /* max_a |r_a - c|^2 */
} tri_geom;

static void tri_geometry(const double *V, const int32_t *F, int64_t k, tri_geom *t)
{
    for (int a = 0; a < 3; ++a)
        for (int d = 0; d < 3; ++d) t->r[a][d] = V[3 * (int64_t)F[3 * k + a] + d];
    double e1[3], e2[3], cr[3];
    sub3(t->r[1], t->r[0], e1);
    sub3(t->r[2], t->r[0], e2);
    cross3(e1, e2, cr);
    double nn = sqrt(dot3(cr, cr));
    t->A = 0.5 * nn;
    for (int d = 0; d < 3; ++d) t->N[d] = cr[d] / nn;
    for (int g = 0; g < 3; ++g)
        for (int d = 0; d < 3; ++d)
            t->y[g][d] = G3_LAMBDA[g][0] * t->r[0][d] + G3_LAMBDA[g][1] * t->r[1][d] + G3_LAMBDA[g][2] * t->r[2][d];
    for (int d = 0; d < 3; ++d) t->c[d] = (t->r[0][d] + t->r[1][d] + t->r[2][d]) / 3.0;
    t->d2 = 0.0;
    for (int a = 0; a < 3; ++a) {
        double v[3];
        sub3(t->r[a], t->c, v);
        double q = dot3(v, v);
        if (q > t->d2) t->d2 = q;
    }
}

/* 3-point Gauss value of  int lambda_a G  and  int lambda_a dG/dn  (SURVEY.md C1,
 * "regular part"): coefficients that multiply q and phi at the triangle's vertices. */
static void gauss3_coeffs(const tri_geom *t, const double *x, double cS[3], double cD[3])
{
    cS[0] = cS[1] = cS[2] = 0.0;
    cD[0] = cD[1] = cD[2] = 0.0;
    double w = t->A / 3.0;
    for (int g = 0; g < 3; ++g) {
        double dx[3];
        sub3(x, t->y[g], dx);
        double rho2 = dot3(dx, dx);
        double rho = sqrt(rho2);
        double kS = w / (FOUR_PI * rho);
        double kD = w * dot3(t->N, dx) / (FOUR_PI * rho2 * rho);
        for (int a = 0; a < 3; ++a) {
            cS[a] += G3_LAMBDA[g][a] * kS;
            cD[a] += G3_LAMBDA[g][a] * kD;
        }
    }
}

/* ------------------------------------------------------------------ */
/* exact flat-triangle integrals of lambda_a G and lambda_a dG/dn       */
/*                                                        */
/* ------------------------------------------------------------------ */

/* collapsed tensor Gauss-Legendre 8x8 on the sub-triangle (p0,p1,p2) whose
 * corners carry barycentric coordinates (b0,b1,b2) of the ROOT triangle.
 * out[0..2] = int lambda_a /(4 pi r),  out[3..5] = int lambda_a N.(x-y)/(4 pi r^3),
 * out[6] = int 1/(4 pi r), out[7] = int 1/(4 pi r^2)  (scales for the tolerance). */
static void subtri_rule(const double p0[3], const double p1[3], const double p2[3],
                        const double b0[3], const double b1[3], const double b2[3],
                        const double N[3], const double x[3], double out[8])
{
    double e1[3], e2[3], cr[3];
    sub3(p1, p0, e1);
    sub3(p2, p0, e2);
    cross3(e1, e2, cr);
    double twoA = sqrt(dot3(cr, cr));
    for (int i = 0; i < 8; ++i) out[i] = 0.0;
    for (int i = 0; i < GL_SMALL; ++i) {
        double s = gl8_x[i];
        for (int j = 0; j < GL_SMALL; ++j) {
            double tt = gl8_x[j];
            double wgt = gl8_w[i] * gl8_w[j] * s * twoA;   /* Jacobian of y = p0 + s[(1-t)e1 + t e2] */
            double c1 = s * (1.0 - tt), c2 = s * tt, c0 = 1.0 - s;
            double y[3], lam[3], dx[3];
            for (int d = 0; d < 3; ++d) {
                y[d] = c0 * p0[d] + c1 * p1[d] + c2 * p2[d];
                lam[d] = c0 * b0[d] + c1 * b1[d] + c2 * b2[d];
            }
            sub3(x, y, dx);
            double r2 = dot3(dx, dx);
            double r = sqrt(r2);
            double kS = wgt / (FOUR_PI * r);
            double kD = wgt * dot3(N, dx) / (FOUR_PI * r2 * r);
            for (int a = 0; a < 3; ++a) {
                out[a] += lam[a] * kS;
                out[3 + a] += lam[a] * kD;
            }
            out[6] += kS;
            out[7] += wgt / (FOUR_PI * r2);
        }
    }
}

static void adapt_rec(const double p0[3], const double p1[3], const double p2[3],
                      const double b0[3], const double b1[3], const double b2[3],
                      const double N[3], const double x[3], const double parent[8],
                      double tolS, double tolD, int depth, double acc[6])
{
    double m01[3], m12[3], m20[3], c01[3], c12[3], c20[3];
    for (int d = 0; d < 3; ++d) {
        m01[d] = 0.5 * (p0[d] + p1[d]); m12[d] = 0.5 * (p1[d] + p2[d]); m20[d] = 0.5 * (p2[d] + p0[d]);
        c01[d] = 0.5 * (b0[d] + b1[d]); c12[d] = 0.5 * (b1[d] + b2[d]); c20[d] = 0.5 * (b2[d] + b0[d]);
    }
    double ch[4][8];
    subtri_rule(p0, m01, m20, b0, c01, c20, N, x, ch[0]);
    subtri_rule(p1, m12, m01, b1, c12, c01, N, x, ch[1]);
    subtri_rule(p2, m20, m12, b2, c20, c12, N, x, ch[2]);
    subtri_rule(m01, m12, m20, c01, c12, c20, N, x, ch[3]);
    int ok = 1;
    for (int a = 0; a < 6; ++a) {
        double sum = ch[0][a] + ch[1][a] + ch[2][a] + ch[3][a];
        double tol = (a < 3) ? tolS : tolD;
        if (fabs(sum - parent[a]) > tol) ok = 0;
    }
    if (ok || depth >= 12) {
        for (int a = 0; a < 6; ++a) acc[a] += ch[0][a] + ch[1][a] + ch[2][a] + ch[3][a];
        return;
    }
    adapt_rec(p0, m01, m20, b0, c01, c20, N, x, ch[0], tolS, tolD, depth + 1, acc);
    adapt_rec(p1, m12, m01, b1, c12, c01, N, x, ch[1], tolS, tolD, depth + 1, acc);
    adapt_rec(p2, m20, m12, b2, c20, c12, N, x, ch[2], tolS, tolD, depth + 1, acc);
    adapt_rec(m01, m12, m20, c01, c12, c20, N, x, ch[3], tolS, tolD, depth + 1, acc);
}

/* x not a vertex of the triangle: recursive 1->4 subdivision, accept a node when
 * the sum of its four children differs from it by < 1e-15 of the root scale. */
static void exact_weights_regular(const tri_geom *t, const double *x, double WS[3], double WD[3])
{
    static const double B0[3] = {1, 0, 0}, B1[3] = {0, 1, 0}, B2[3] = {0, 0, 1};
    double root[8], acc[6] = {0, 0, 0, 0, 0, 0};
    subtri_rule(t->r[0], t->r[1], t->r[2], B0, B1, B2, t->N, x, root);
    adapt_rec(t->r[0], t->r[1], t->r[2], B0, B1, B2, t->N, x, root,
              1e-15 * root[6], 1e-15 * root[7], 0, acc);
    for (int a = 0; a < 3; ++a) { WS[a] = acc[a]; WD[a] = acc[3 + a]; }
}

/* x == vertex a0 of the triangle: W^D = 0 exactly (x lies in the plane); W^S by
 * the Duffy collapse y = x + u[(1-v)a + v b], composite 4 x 32-point
 * Gauss-Legendre in v for I0 = int dv/|e(v)|, I1 = int v dv/|e(v)|. */
static void exact_weights_incident(const tri_geom *t, int a0, double WS[3], double WD[3])
{
    const double *x = t->r[a0];
    double a[3], b[3];
    sub3(t->r[(a0 + 1) % 3], x, a);
    sub3(t->r[(a0 + 2) % 3], x, b);
    double I0 = 0.0, I1 = 0.0;
    const int panels = 4;
    for (int pnl = 0; pnl < panels; ++pnl) {
        for (int i = 0; i < GL_BIG; ++i) {
            double v = (pnl + gl32_x[i]) / panels;
            double w = gl32_w[i] / panels;
            double e[3];
            for (int d = 0; d < 3; ++d) e[d] = a[d] + v * (b[d] - a[d]);
            double inv = 1.0 / sqrt(dot3(e, e));
            I0 += w * inv;
            I1 += w * v * inv;
        }
    }
    double f = 2.0 * t->A / FOUR_PI * 0.5;
    WS[a0] = f * I0;
    WS[(a0 + 1) % 3] = f * (I0 - I1);
    WS[(a0 + 2) % 3] = f * I1;
    WD[0] = WD[1] = WD[2] = 0.0;
}

/* exported for the pins: exact weights of one triangle seen from x.
 * incident_local = local index (0..2) of the vertex equal to x, or -1. */
void oracle_exact_weights(const double *tri9, const double *x, int incident_local,
                          double *WS, double *WD)
{
    gl_init();
    double V[9];
    int32_t F[3] = {0, 1, 2};
    memcpy(V, tri9, sizeof V);
    tri_geom t;
    tri_geometry(V, F, 0, &t);
    if (incident_local >= 0) exact_weights_incident(&t, incident_local, WS, WD);
    else exact_weights_regular(&t, x, WS, WD);
}

/* exported for the pins: the 3-point Gauss coefficients of one triangle */
void oracle_gauss3_coeffs(const double *tri9, const double *x, double *cS, double *cD)
{
    double V[9];
    int32_t F[3] = {0, 1, 2};
    memcpy(V, tri9, sizeof V);
    tri_geom t;
    tri_geometry(V, F, 0, &t);
    gauss3_coeffs(&t, x, cS, cD);
}

/* ------------------------------------------------------------------ */
/* mode G3: coefficients of (q, phi) at the vertices of triangle k for  */
/* collocation vertex i                                  */
/* ------------------------------------------------------------------ */
static int g3_tri_coeffs(const double *V, const int32_t *F, int64_t i, int64_t k, double eta,
                         double cS[3], double cD[3])
{
    tri_geom t;
    tri_geometry(V, F, k, &t);
    const double *x = V + 3 * i;
    gauss3_coeffs(&t, x, cS, cD);
    int inc = -1;
    for (int a = 0; a < 3; ++a)
        if ((int64_t)F[3 * k + a] == i) inc = a;
    double dc[3];
    sub3(x, t.c, dc);
    int near = (inc >= 0) || (dot3(dc, dc) <= eta * eta * t.d2);
    if (!near) return 0;
    double WS[3], WD[3];
    if (inc >= 0) exact_weights_incident(&t, inc, WS, WD);
    else exact_weights_regular(&t, x, WS, WD);
    /* the correction (W - Gauss) added to the Gauss value leaves W */
    for (int a = 0; a < 3; ++a) { cS[a] = WS[a]; cD[a] = WD[a]; }
    return 1;
}

/* y[r] = (S q - D phi)(rows[r]);  q or phi may be NULL (zero density).
 * near_count (optional, may be NULL): number of near triangles of each row. */
int oracle_g3_apply_rows(const double *V, int64_t N, const int32_t *F, int64_t T,
                         const double *q, const double *phi, double eta,
                         const int64_t *rows, int64_t nrows, double *y, int64_t *near_count)
{
    (void)N;
    gl_init();
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nrows; ++r) {
        int64_t i = rows[r];
        ksum acc = {0.0, 0.0};
        int64_t nn = 0;
        for (int64_t k = 0; k < T; ++k) {
            double cS[3], cD[3];
            nn += g3_tri_coeffs(V, F, i, k, eta, cS, cD);
            double v = 0.0;
            for (int a = 0; a < 3; ++a) {
                int64_t j = F[3 * k + a];
                if (q) v += cS[a] * q[j];
                if (phi) v -= cD[a] * phi[j];
            }
            ksum_add(&acc, v);
        }
        y[r] = ksum_get(&acc);
        if (near_count) near_count[r] = nn;
    }
    return 0;
}

/* dense rows of the matrices: S[r*N + j], D[r*N + j]  (tiny meshes only) */
int oracle_g3_dense_rows(const double *V, int64_t N, const int32_t *F, int64_t T, double eta,
                         const int64_t *rows, int64_t nrows, double *S, double *D)
{
    gl_init();
    memset(S, 0, sizeof(double) * (size_t)(nrows * N));
    memset(D, 0, sizeof(double) * (size_t)(nrows * N));
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nrows; ++r) {
        int64_t i = rows[r];
        for (int64_t k = 0; k < T; ++k) {
            double cS[3], cD[3];
            g3_tri_coeffs(V, F, i, k, eta, cS, cD);
            for (int a = 0; a < 3; ++a) {
                int64_t j = F[3 * k + a];
                S[r * N + j] += cS[a];
                D[r * N + j] += cD[a];
            }
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* mode V1: the paper's lumped quadrature (Eq. 17) + diagonal (19-21)   */
/* ------------------------------------------------------------------ */

/* s_j = 1/3 sum_{k ni j} A_k ;  n_j = m_j/|m_j|, m_j = sum_{k ni j} N_k A_k */
int oracle_v1_vertex_weights(const double *V, int64_t N, const int32_t *F, int64_t T,
                             double *s, double *n)
{
    memset(s, 0, sizeof(double) * (size_t)N);
    memset(n, 0, sizeof(double) * (size_t)(3 * N));
    for (int64_t k = 0; k < T; ++k) {
        tri_geom t;
        tri_geometry(V, F, k, &t);
        for (int a = 0; a < 3; ++a) {
            int64_t j = F[3 * k + a];
            s[j] += t.A / 3.0;
            for (int d = 0; d < 3; ++d) n[3 * j + d] += t.N[d] * t.A;
        }
    }
    for (int64_t j = 0; j < N; ++j) {
        double nn = sqrt(dot3(n + 3 * j, n + 3 * j));
        for (int d = 0; d < 3; ++d) n[3 * j + d] /= nn;
    }
    return 0;
}

/* y[r] = sum_j L_ij q_j - M_ij phi_j with
 *   L_ij = s_j /(4 pi |r_i - r_j|),  M_ij = s_j n_j.(r_i - r_j)/(4 pi |r_i - r_j|^3),  i != j
 *   M_ii = -1/2 - sum_{j != i} M_ij
 *   L_ii = n_i . sum_{j != i} [ M_ij (r_j - r_i) - L_ij n_j ]         (Eq. 21, PAPER.md:214,
 *          written in its translation-invariant form: substitute M_ii into Eq. 21)
 * Ldiag / Mdiag (optional) receive the diagonal entries of the rows. */
int oracle_v1_apply_rows(const double *V, int64_t N, const int32_t *F, int64_t T,
                         const double *q, const double *phi,
                         const int64_t *rows, int64_t nrows, double *y,
                         double *Ldiag, double *Mdiag)
{
    double *s = (double *)malloc(sizeof(double) * (size_t)N);
    double *n = (double *)malloc(sizeof(double) * (size_t)(3 * N));
    if (!s || !n) { free(s); free(n); return 1; }
    oracle_v1_vertex_weights(V, N, F, T, s, n);
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nrows; ++r) {
        int64_t i = rows[r];
        const double *x = V + 3 * i;
        ksum acc = {0, 0}, msum = {0, 0}, lv[3] = {{0, 0}, {0, 0}, {0, 0}};
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            double dx[3];
            sub3(x, V + 3 * j, dx);
            double r2 = dot3(dx, dx);
            double rr = sqrt(r2);
            double Lij = s[j] / (FOUR_PI * rr);
            double Mij = s[j] * dot3(n + 3 * j, dx) / (FOUR_PI * r2 * rr);
            double v = 0.0;
            if (q) v += Lij * q[j];
            if (phi) v -= Mij * phi[j];
            ksum_add(&acc, v);
            ksum_add(&msum, Mij);
            for (int d = 0; d < 3; ++d) ksum_add(&lv[d], Mij * (-dx[d]) - Lij * n[3 * j + d]);
        }
        double Mii = -0.5 - ksum_get(&msum);
        double Lii = 0.0;
        for (int d = 0; d < 3; ++d) Lii += n[3 * i + d] * ksum_get(&lv[d]);
        double v = ksum_get(&acc);
        if (q) v += Lii * q[i];
        if (phi) v -= Mii * phi[i];
        y[r] = v;
        if (Ldiag) Ldiag[r] = Lii;
        if (Mdiag) Mdiag[r] = Mii;
    }
    free(s);
    free(n);
    return 0;
}

/* ------------------------------------------------------------------ */
/* point sums used by the engine-level pins (Table 1 workload):         */
/* y[r] = sum_j m_j / (4 pi |x_r - y_j|), skipping coincident points     */
/* ------------------------------------------------------------------ */
int oracle_monopole_sum(const double *src, const double *m, int64_t ns,
                        const double *tgt, int64_t nt, double *y)
{
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < nt; ++r) {
        ksum acc = {0, 0};
        for (int64_t j = 0; j < ns; ++j) {
            double dx[3];
            sub3(tgt + 3 * r, src + 3 * j, dx);
            double r2 = dot3(dx, dx);
            if (r2 == 0.0) continue;
            ksum_add(&acc, m[j] / (FOUR_PI * sqrt(r2)));
        }
        y[r] = ksum_get(&acc);
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* point sums with dipoles (Eq. 13: G and dG/dn with   */
/* the normal folded into the dipole strength d_j):                     */
/* y[r] = sum_j [ m_j / (4 pi |x_r - y_j|)                              */
/*              - d_j . (x_r - y_j) / (4 pi |x_r - y_j|^3) ],           */
/* coincident points skipped; m or d may be NULL (zero strengths).      */
/* With m_j = q_j w_j and d_j = phi_j n_j w_j this is the quadrature of */
/* S[q] - D[phi] over points y_j with weights w_j and normals n_j.      */
/* ------------------------------------------------------------------ */
int oracle_point_sum(const double *src, const double *m, const double *d, int64_t ns,
                     const double *tgt, int64_t nt, double *y)
{
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < nt; ++r) {
        ksum acc = {0, 0};
        for (int64_t j = 0; j < ns; ++j) {
            double dx[3];
            sub3(tgt + 3 * r, src + 3 * j, dx);
            double r2 = dot3(dx, dx);
            if (r2 == 0.0) continue;
            double rr = sqrt(r2);
            double v = 0.0;
            if (m) v += m[j] / (FOUR_PI * rr);
            if (d) v -= dot3(d + 3 * j, dx) / (FOUR_PI * r2 * rr);
            ksum_add(&acc, v);
        }
        y[r] = ksum_get(&acc);
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* mode G3 at points OFF the surface (Eq. 11, the cases   */
/* r not on S): u(x) = S[q](x) - D[phi](x) with the same discretisation */
/* as at the vertices -- 3-point Gauss per triangle with */
/* P1 densities, and the exact flat-triangle integrals on the near set  */
/* { k : |x - c_k| <= eta d_k }.  No triangle is incident to x.         */
/* ------------------------------------------------------------------ */
int oracle_g3_evaluate(const double *V, int64_t N, const int32_t *F, int64_t T,
                       const double *q, const double *phi, double eta,
                       const double *X, int64_t nx, double *y, int64_t *near_count)
{
    (void)N;
    gl_init();
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nx; ++r) {
        const double *x = X + 3 * r;
        ksum acc = {0.0, 0.0};
        int64_t nn = 0;
        for (int64_t k = 0; k < T; ++k) {
            tri_geom t;
            tri_geometry(V, F, k, &t);
            double cS[3], cD[3];
            gauss3_coeffs(&t, x, cS, cD);
            double dc[3];
            sub3(x, t.c, dc);
            if (dot3(dc, dc) <= eta * eta * t.d2) {
                exact_weights_regular(&t, x, cS, cD);
                ++nn;
            }
            double v = 0.0;
            for (int a = 0; a < 3; ++a) {
                int64_t j = F[3 * k + a];
                if (q) v += cS[a] * q[j];
                if (phi) v -= cD[a] * phi[j];
            }
            ksum_add(&acc, v);
        }
        y[r] = ksum_get(&acc);
        if (near_count) near_count[r] = nn;
    }
    return 0;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
