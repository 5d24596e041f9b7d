/*
 * mesh_ft_oracle.c -- fp64 CPU ORACLE for the mesh Fourier transform of deltaMic (arxiv 2303.10440).
 *
 * THIS IS TEST INFRASTRUCTURE.  It defines what the CUDA path must compute and is imported only by
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.  It shares no
 * code, header, table or helper with paper_2303_10440_b200/csrc and is never on the product path.
 * Plain, slow, written to be checked against the paper by eye; never tuned.
 *
 * What it computes (PAPER.md line numbers refer to /root/reference/PAPER.md):
 *
 *   surface mode  F(k) = sum_T  int_T exp(-i k.x) dS = sum_T 2 A_T f_T(k)      PAPER.md:156-163 eq. 8-9,
 *                                                                              :177-180 eq. 12 without
 *                                                                              the 1/|Lambda| (reading R7)
 *   volume  mode  F(k) = int_Omega exp(-i k.x) d^3x
 *                      = (i/|k|^2) sum_T (k.m_T) f_T(k),  F(0) = 1/6 sum_T v1.(v2 x v3)
 *                      (divergence theorem with the field i k exp(-i k.x)/|k|^2; BASELINE.json north_star)
 *   gradient      dL/dv = sum_k Re( conj(G(k)) dF(k)/dv ),  G = dL/dRe F + i dL/dIm F   (reading R14),
 *                 summed over the vertex star (eq. 13).
 *
 * with a = k.v1, b = k.v2, c = k.v3,  m_T = (v2-v1) x (v3-v1) = 2 A_T N_T,  and
 *
 *   f_T(k) = g(a,b,c) = int_{t1,t2>=0, t1+t2<=1} exp(-i(a + t1 (b-a) + t2 (c-a))) dt1 dt2
 *          = exp[-ia, -ib, -ic]      (second divided difference of exp)
 *          = eq. 9 / eq. 14 of the paper away from coincident arguments (readings R1, R3), and
 *          = eq. 15 / eq. 16 in the confluent limits.
 *
 * The paper evaluates eq. 9 and switches to the zeroth-order limits eq. 15/16 below an unstated
 * threshold eps, which leaves an O(eps) error (reading R4).  The method reaches an
 * exactly defined quantity (the integral), so the oracle evaluates THAT: divided differences of exp
 * computed by the textbook recursion when the nodes are separated and by the (exact, convergent)
 * power series in the centred nodes when they cluster (step O2).  No blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_*.py): analytic box product-of-sincs (P1), F(0) = volume / area (P2),
 * translation/scaling/orientation identities (P3), eq. 9 / 15 / 16 in 50-digit arithmetic (P4),
 * Gauss quadrature per triangle (P5), voxelised-indicator DFT (P6), ball / shell closed forms (P7),
 * central finite differences (P8), exact gradient identities (P9).
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (oracle/build.py).  No -ffast-math.
 */
#include <complex.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#define DD_CLUSTER_DIAMETER 0.5 /* step O2: series when all nodes lie within this diameter */
#define DD_MAX_TERMS 60

/* Divided difference of exp on n <= 4 clustered complex nodes, by its power series:
 *   exp[z_0..z_{n-1}] = e^mu * sum_{m>=0} h_m(z - mu) / (m + n - 1)!
 * h_m = complete homogeneous symmetric polynomial of degree m, from Newton's recurrence
 *   h_m = e_1 h_{m-1} - e_2 h_{m-2} + e_3 h_{m-3} - e_4 h_{m-4},   e_j elementary symmetric. */
static cplx dd_exp_series(const cplx *z, int n)
{
    cplx mu = 0.0;
    for (int i = 0; i < n; ++i) mu += z[i];
    mu /= (double)n;
    cplx e[5] = {1.0, 0.0, 0.0, 0.0, 0.0};
    for (int i = 0; i < n; ++i) {
        cplx w = z[i] - mu;
        for (int j = n; j >= 1; --j) e[j] += e[j - 1] * w;
    }
    cplx h[DD_MAX_TERMS];
    double fact = 1.0; /* (m + n - 1)! */
    for (int j = 2; j <= n - 1; ++j) fact *= (double)j;
    cplx sum = 0.0;
    int small = 0;
    for (int m = 0; m < DD_MAX_TERMS; ++m) {
        if (m == 0) {
            h[0] = 1.0;
        } else {
            cplx acc = 0.0;
            double sign = 1.0;
            for (int j = 1; j <= n && j <= m; ++j) {
                acc += sign * e[j] * h[m - j];
                sign = -sign;
            }
            h[m] = acc;
            fact *= (double)(m + n - 1);
        }
        cplx term = h[m] / fact;
        sum += term;
        /* stop after two consecutive negligible terms (one term alone can vanish by symmetry) */
        small = (cabs(term) < 1e-20) ? small + 1 : 0;
        if (small >= 2) break;
    }
    return cexp(mu) * sum;
}

/* Divided difference of exp on n <= 4 complex nodes (repeated nodes allowed).
 * Separated nodes: f[Z] = (f[Z \ z_j] - f[Z \ z_i]) / (z_i - z_j) on the farthest pair (i, j), so every
 * division is by a number >= DD_CLUSTER_DIAMETER in modulus.  Clustered nodes: the series above. */
static cplx dd_exp(const cplx *z, int n)
{
    if (n == 1) return cexp(z[0]);
    double dmax = -1.0;
    int bi = 0, bj = 1;
    for (int i = 0; i < n; ++i)
        for (int j = i + 1; j < n; ++j) {
            double d = cabs(z[i] - z[j]);
            if (d > dmax) { dmax = d; bi = i; bj = j; }
        }
    if (dmax < DD_CLUSTER_DIAMETER) return dd_exp_series(z, n);
    cplx without_i[3], without_j[3];
    int ni = 0, nj = 0;
    for (int q = 0; q < n; ++q) {
        if (q != bi) without_i[ni++] = z[q];
        if (q != bj) without_j[nj++] = z[q];
    }
    return (dd_exp(without_j, n - 1) - dd_exp(without_i, n - 1)) / (z[bi] - z[bj]);
}

/* g(a,b,c) of the header = f_T (PAPER.md:162 eq. 9, :194 eq. 14 with readings R1/R3). */
static cplx g_fun(double a, double b, double c)
{
    cplx z[3] = {-I * a, -I * b, -I * c};
    return dd_exp(z, 3);
}

/* dg/da_p, p = 0,1,2: differentiating a divided difference wrt a node repeats that node;
 * the node is -i a_p, hence the factor -i.  (Exact counterpart of PAPER.md:171-173 eq. 11, R2.) */
static void g_grad(double a, double b, double c, cplx dg[3])
{
    double x[3] = {a, b, c};
    for (int p = 0; p < 3; ++p) {
        cplx z[4] = {-I * x[0], -I * x[1], -I * x[2], -I * x[p]};
        dg[p] = -I * dd_exp(z, 4);
    }
}

static inline void cross3(const double *u, const double *v, double *o)
{
    o[0] = u[1] * v[2] - u[2] * v[1];
    o[1] = u[2] * v[0] - u[0] * v[2];
    o[2] = u[0] * v[1] - u[1] * v[0];
}
static inline double dot3(const double *u, const double *v) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; }

/* ---- exported test hooks for pin P4 ------------------------------------------------------- */
void oracle_g(double a, double b, double c, double *out2)
{
    cplx g = g_fun(a, b, c);
    out2[0] = creal(g);
    out2[1] = cimag(g);
}
void oracle_g_grad(double a, double b, double c, double *out6)
{
    cplx dg[3];
    g_grad(a, b, c, dg);
    for (int p = 0; p < 3; ++p) { out6[2 * p] = creal(dg[p]); out6[2 * p + 1] = cimag(dg[p]); }
}
int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- forward (steps O1, O3) ---------------------------------------------------------------
 * vertices [n_v*3] fp64 (the fp32 inputs promoted, R21), faces [n_f*3] int32, kvec [n_k*3] angular
 * frequencies, mode 0 = volume / 1 = surface, F_out [n_k] complex interleaved.  Returns 0, or -1 on a
 * bad argument / face index. */
int oracle_mesh_ft_forward(const double *vertices, int32_t n_v, const int32_t *faces, int32_t n_f,
                           const double *kvec, int64_t n_k, int32_t mode, double *F_out)
{
    if (!vertices || !faces || !kvec || !F_out || n_v < 0 || n_f < 0 || n_k < 0 || (mode != 0 && mode != 1)) return -1;
    for (int64_t t = 0; t < (int64_t)n_f * 3; ++t)
        if (faces[t] < 0 || faces[t] >= n_v) return -1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t q = 0; q < n_k; ++q) {
        const double *k = kvec + 3 * q;
        const double k2 = dot3(k, k);
        cplx acc = 0.0;
        for (int32_t t = 0; t < n_f; ++t) {
            const double *v1 = vertices + 3 * (size_t)faces[3 * t + 0];
            const double *v2 = vertices + 3 * (size_t)faces[3 * t + 1];
            const double *v3 = vertices + 3 * (size_t)faces[3 * t + 2];
            double u[3] = {v2[0] - v1[0], v2[1] - v1[1], v2[2] - v1[2]};
            double w[3] = {v3[0] - v1[0], v3[1] - v1[1], v3[2] - v1[2]};
            double m[3];
            cross3(u, w, m); /* m_T = 2 A_T N_T */
            if (mode == 1) { /* surface: 2 A_T g  (eq. 8) */
                acc += sqrt(dot3(m, m)) * g_fun(dot3(k, v1), dot3(k, v2), dot3(k, v3));
            } else if (k2 == 0.0) { /* volume, k = 0: signed tetrahedron */
                double c23[3];
                cross3(v2, v3, c23);
                acc += dot3(v1, c23) / 6.0;
            } else { /* volume: (i/|k|^2)(k.m_T) g */
                acc += (I / k2) * dot3(k, m) * g_fun(dot3(k, v1), dot3(k, v2), dot3(k, v3));
            }
        }
        F_out[2 * q] = creal(acc);
        F_out[2 * q + 1] = cimag(acc);
    }
    return 0;
}

/* ---- backward (steps O4, O5, O6) ------------------------------------------------------------
 * G [n_k] complex interleaved = dL/dRe F + i dL/dIm F on exactly the listed frequencies (R14);
 * dL_dv [n_v*3] overwritten.  corner_scratch [n_f*9] receives the per-corner gradients (may be NULL).
 *
 * surface (eq. 10):  d(2A g)/dv_p = -w_p g + 2A k dg/da_p,  w_p = e_p x N_T,
 *                                     e_p = v_{p-} - v_{p+}, zero-area triangle -> 0 (R19)
 * volume  (product rule, O4):         dF/dv_p|_T = (i/|k|^2)[(k x e_p) g + (k.m_T) k dg/da_p],
 *                                     k = 0:  dV/dv_p|_T = (v_{p+} x v_{p-})/6. */
int oracle_mesh_ft_backward(const double *vertices, int32_t n_v, const int32_t *faces, int32_t n_f,
                            const double *kvec, int64_t n_k, int32_t mode, const double *G,
                            double *dL_dv, double *corner_scratch)
{
    if (!vertices || !faces || !kvec || !G || !dL_dv || n_v < 0 || n_f < 0 || n_k < 0 || (mode != 0 && mode != 1)) return -1;
    for (int64_t t = 0; t < (int64_t)n_f * 3; ++t)
        if (faces[t] < 0 || faces[t] >= n_v) return -1;
    for (int64_t i = 0; i < (int64_t)n_v * 3; ++i) dL_dv[i] = 0.0;
    double *corner = corner_scratch ? corner_scratch : (double *)malloc(sizeof(double) * 9 * (size_t)(n_f > 0 ? n_f : 1));
    if (!corner) return -2;

#pragma omp parallel for schedule(dynamic, 4)
    for (int32_t t = 0; t < n_f; ++t) {
        const double *v[3] = {vertices + 3 * (size_t)faces[3 * t + 0], vertices + 3 * (size_t)faces[3 * t + 1],
                              vertices + 3 * (size_t)faces[3 * t + 2]};
        double e[3][3]; /* e_p = v_{p-} - v_{p+} */
        for (int p = 0; p < 3; ++p) {
            const double *vm = v[(p + 2) % 3], *vp = v[(p + 1) % 3];
            for (int d = 0; d < 3; ++d) e[p][d] = vm[d] - vp[d];
        }
        double m[3];
        cross3(e[2], e[0], m); /* e_3 x e_1 = 2 A N */
        const double mnorm = sqrt(dot3(m, m));
        double grad[3][3] = {{0}};
        double wv[3][3] = {{0}};
        if (mode == 1 && mnorm >= 1e-30) {
            double N[3] = {m[0] / mnorm, m[1] / mnorm, m[2] / mnorm};
            for (int p = 0; p < 3; ++p) cross3(e[p], N, wv[p]);
        }
        for (int64_t q = 0; q < n_k; ++q) {
            const double *k = kvec + 3 * q;
            const cplx Gc = conj(G[2 * q] + I * G[2 * q + 1]);
            const double k2 = dot3(k, k);
            if (mode == 1) {
                if (mnorm < 1e-30) continue;
                cplx g = g_fun(dot3(k, v[0]), dot3(k, v[1]), dot3(k, v[2]));
                cplx dg[3];
                g_grad(dot3(k, v[0]), dot3(k, v[1]), dot3(k, v[2]), dg);
                const double s0 = creal(Gc * g);
                for (int p = 0; p < 3; ++p) {
                    const double sp = creal(Gc * dg[p]);
                    for (int d = 0; d < 3; ++d) grad[p][d] += -wv[p][d] * s0 + mnorm * k[d] * sp;
                }
            } else if (k2 == 0.0) {
                for (int p = 0; p < 3; ++p) {
                    double c[3];
                    cross3(v[(p + 1) % 3], v[(p + 2) % 3], c);
                    for (int d = 0; d < 3; ++d) grad[p][d] += creal(Gc) * c[d] / 6.0;
                }
            } else {
                cplx g = g_fun(dot3(k, v[0]), dot3(k, v[1]), dot3(k, v[2]));
                cplx dg[3];
                g_grad(dot3(k, v[0]), dot3(k, v[1]), dot3(k, v[2]), dg);
                const cplx chi = Gc * I / k2;
                const double km = dot3(k, m);
                const double s0 = creal(chi * g);
                for (int p = 0; p < 3; ++p) {
                    double kxe[3];
                    cross3(k, e[p], kxe);
                    const double sp = creal(chi * dg[p]);
                    for (int d = 0; d < 3; ++d) grad[p][d] += kxe[d] * s0 + km * k[d] * sp;
                }
            }
        }
        for (int p = 0; p < 3; ++p)
            for (int d = 0; d < 3; ++d) corner[9 * (size_t)t + 3 * p + d] = grad[p][d];
    }
    /* step O6: scatter over the vertex star (eq. 13), serially, in face order (deterministic) */
    for (int32_t t = 0; t < n_f; ++t)
        for (int p = 0; p < 3; ++p)
            for (int d = 0; d < 3; ++d) dL_dv[3 * (size_t)faces[3 * t + p] + d] += corner[9 * (size_t)t + 3 * p + d];
    if (!corner_scratch) free(corner);
    return 0;
}
