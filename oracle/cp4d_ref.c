/*
 * oracle/cp4d_ref.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what the cp4d hot path computes: the discrete operators
 * K1 (time-decomposed parallel-beam projector), K1^T, K2 = grad_{lambda2}, div = -K2^T, the two
 * dual proxes, the Chambolle-Pock loop of PAPER.md Fig. 2 (L147-L168) and the power iteration
 * for ||K||.  Written from PAPER.md and the readings listed in DESIGN.md ("Readings"); shares no
 * code, header, table or constant with the CUDA path under paper_1809_09725_b200/csrc/.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * load this library.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): dense brute-force K on 8x8 grids, theta=0
 * and pi/2 reduce to column/row sums, ray-stepping forward vs closed-form hat matrix, adjoint
 * dot-product identity, div = -grad^T, closed-form ||K2||^2, closed-form Radon transform of a
 * disk and a Gaussian, pi-symmetry (fold), Moreau identity for the F2* prox, optimality residual
 * of the F1* prox, power iteration vs dense SVD, KKT / Fejer / lambda1=0 checks of the CP loop.
 * No function here is "parity unpinned".
 *
 * Layouts (identical to include/cp4d.h so buffers compare element by element):
 *   primal-shaped  f[z][iy][ix][j]          j fastest, size nz*n*n*m
 *   sinogram       g[z][k][b]               b fastest, size nz*n_angles*nd
 *   dual field     p[a][z][iy][ix][j]       a = 0..3 = (x, y, z, t), component-major
 *   basis table    phi[j][k] = phi_j(t_k)   size m*n_angles
 * Geometry (R1/R2): voxel centres x = ix-(n-1)/2, y = iy-(n-1)/2; bins s_b = b-(nd-1)/2;
 *   theta_k = k*pi/n_theta0 with n_theta0 = n_angles/n_half_rot; a_k = max(|cos|,|sin|).
 *
 * Threads: every output element is summed by exactly one thread in a fixed order, so results
 * are bitwise independent of the thread count; the definition is nthreads = 1
 * (cp4d_ref_set_threads), more threads are the "fast oracle" of DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PI 3.14159265358979323846264338327950288

typedef struct {
    int32_t n, nz, nd, n_angles, n_half_rot, m;
    double lambda1, lambda2;
    const double *phi; /* m * n_angles */
} ref_prob;

static int g_threads = 1;
void cp4d_ref_set_threads(int t) { g_threads = t < 1 ? 1 : t; }
int cp4d_ref_get_threads(void) { return g_threads; }
int cp4d_ref_max_threads(void) {
#ifdef _OPENMP
    return omp_get_num_procs();
#else
    return 1;
#endif
}

static inline int64_t V_of(const ref_prob *P) { return (int64_t)P->nz * P->n * P->n * P->m; }
static inline int64_t S_of(const ref_prob *P) { return (int64_t)P->nz * P->n_angles * P->nd; }
int64_t cp4d_ref_V(const ref_prob *P) { return V_of(P); }
int64_t cp4d_ref_S(const ref_prob *P) { return S_of(P); }

static inline double theta_of(const ref_prob *P, int k) {
    return (double)k * PI / (double)(P->n_angles / P->n_half_rot);
}

/* ---------------------------------------------------------------------------------------------
 * O1/O2  Joseph ray sum of one ray (z, angle (c,s), bin b) for all m coefficients: acc[j].
 * DESIGN.md reading R3 (the paper's own discretisation, log-polar, is not given: PAPER.md:L281).
 * Steps along the dominant axis, linear interpolation between the two nearest samples on the
 * other axis, scaled by 1/max(|c|,|s|).  Values outside the grid are zero.
 * ------------------------------------------------------------------------------------------- */
static void joseph_ray(const ref_prob *P, const double *fz /* slice z: [iy][ix][j] */, double c, double s,
                       int b, double *acc) {
    const int n = P->n, m = P->m;
    const double cen = 0.5 * (n - 1), sb = (double)b - 0.5 * (P->nd - 1);
    for (int j = 0; j < m; ++j) acc[j] = 0.0;
    if (fabs(s) >= fabs(c)) { /* step over columns ix, interpolate along y */
        for (int ix = 0; ix < n; ++ix) {
            double x = ix - cen;
            double ys = (sb - x * c) / s + cen; /* fractional row index */
            double fl = floor(ys);
            int r = (int)fl;
            double w1 = ys - fl, w0 = 1.0 - w1;
            if (r >= 0 && r < n) {
                const double *v = fz + ((int64_t)r * n + ix) * m;
                for (int j = 0; j < m; ++j) acc[j] += w0 * v[j];
            }
            if (r + 1 >= 0 && r + 1 < n) {
                const double *v = fz + ((int64_t)(r + 1) * n + ix) * m;
                for (int j = 0; j < m; ++j) acc[j] += w1 * v[j];
            }
        }
        for (int j = 0; j < m; ++j) acc[j] /= fabs(s);
    } else { /* step over rows iy, interpolate along x */
        for (int iy = 0; iy < n; ++iy) {
            double y = iy - cen;
            double xs = (sb - y * s) / c + cen;
            double fl = floor(xs);
            int q = (int)fl;
            double w1 = xs - fl, w0 = 1.0 - w1;
            if (q >= 0 && q < n) {
                const double *v = fz + ((int64_t)iy * n + q) * m;
                for (int j = 0; j < m; ++j) acc[j] += w0 * v[j];
            }
            if (q + 1 >= 0 && q + 1 < n) {
                const double *v = fz + ((int64_t)iy * n + q + 1) * m;
                for (int j = 0; j < m; ++j) acc[j] += w1 * v[j];
            }
        }
        for (int j = 0; j < m; ++j) acc[j] /= fabs(c);
    }
}

/* O2  forward, the definition: (K1 f)[z,k,b] = sum_j phi[j,k] * (R_{theta_k} f_j)[b]
 * PAPER.md Eq. 9 (L184) / L231, one Radon transform per angle, no folding. */
void cp4d_ref_forward(const ref_prob *P, const double *f, double *g) {
    const int n = P->n, m = P->m, na = P->n_angles, nd = P->nd;
    const int64_t rows = (int64_t)P->nz * na;
#pragma omp parallel for schedule(dynamic, 4) num_threads(g_threads)
    for (int64_t zk = 0; zk < rows; ++zk) {
        int z = (int)(zk / na), k = (int)(zk % na);
        double th = theta_of(P, k), c = cos(th), s = sin(th);
        double acc[64];
        const double *fz = f + (int64_t)z * n * n * m;
        for (int b = 0; b < nd; ++b) {
            joseph_ray(P, fz, c, s, b, acc);
            double v = 0.0;
            for (int j = 0; j < m; ++j) v += P->phi[(int64_t)j * na + k] * acc[j];
            g[zk * nd + b] = v;
        }
    }
}

/* A8  forward with the paper's pi-folding: R f_j is computed for the base
 * angles theta_0 in [0,pi) only and distributed to k = q*n_theta0 + i with s -> (-1)^q s,
 * which on the symmetric detector is the index flip b -> nd-1-b. */
void cp4d_ref_forward_folded(const ref_prob *P, const double *f, double *g) {
    const int n = P->n, m = P->m, na = P->n_angles, nd = P->nd, n0 = na / P->n_half_rot;
    const int64_t rows = (int64_t)P->nz * n0;
#pragma omp parallel for schedule(dynamic, 2) num_threads(g_threads)
    for (int64_t zi = 0; zi < rows; ++zi) {
        int z = (int)(zi / n0), i = (int)(zi % n0);
        double th = theta_of(P, i), c = cos(th), s = sin(th);
        double acc[64];
        const double *fz = f + (int64_t)z * n * n * m;
        for (int b = 0; b < nd; ++b) {
            joseph_ray(P, fz, c, s, b, acc);
            for (int q = 0; q < P->n_half_rot; ++q) {
                int k = q * n0 + i, bb = (q & 1) ? nd - 1 - b : b;
                double v = 0.0;
                for (int j = 0; j < m; ++j) v += P->phi[(int64_t)j * na + k] * acc[j];
                g[((int64_t)z * na + k) * nd + bb] = v;
            }
        }
    }
}

/* forward at sampled rays (z,k,b) -- O(n*m) each; for parity at sizes the full oracle cannot run */
void cp4d_ref_forward_rays(const ref_prob *P, const double *f, int64_t ns, const int32_t *zkb, double *out) {
    const int n = P->n, m = P->m, na = P->n_angles;
#pragma omp parallel for schedule(dynamic, 16) num_threads(g_threads)
    for (int64_t i = 0; i < ns; ++i) {
        int z = zkb[3 * i], k = zkb[3 * i + 1], b = zkb[3 * i + 2];
        double th = theta_of(P, k), acc[64], v = 0.0;
        joseph_ray(P, f + (int64_t)z * n * n * m, cos(th), sin(th), b, acc);
        for (int j = 0; j < m; ++j) v += P->phi[(int64_t)j * na + k] * acc[j];
        out[i] = v;
    }
}

/* ---------------------------------------------------------------------------------------------
 * O1 closed form: A_k[b; iy,ix] = Lambda((x c + y s - s_b)/a)/a, Lambda(u) = max(0, 1-|u|).
 * O3 adjoint, the definition: (K1^T g)[j,z,iy,ix] = sum_k phi[j,k] sum_b A_k[b;iy,ix] g[z,k,b]
 * (Eq. 10, with phi-hat = phi for a real table).  No pi/N_theta weight, no filter:
 * the exact transpose of O2.  Only b in {floor(p), floor(p)+1} can have a non-zero weight.
 * ------------------------------------------------------------------------------------------- */
static inline double hat_weight(double u, double a) {
    double w = 1.0 - fabs(u) / a;
    return w > 0.0 ? w / a : 0.0;
}

static void adjoint_voxel(const ref_prob *P, const double *gz /* [k][b] of slice z */, int iy, int ix,
                          int k_begin, int k_end, double *acc /* m, accumulated into */) {
    const int n = P->n, m = P->m, na = P->n_angles, nd = P->nd;
    const double x = ix - 0.5 * (n - 1), y = iy - 0.5 * (n - 1), cd = 0.5 * (nd - 1);
    for (int k = k_begin; k < k_end; ++k) {
        double th = theta_of(P, k), c = cos(th), s = sin(th);
        double a = fmax(fabs(c), fabs(s));
        double p = x * c + y * s + cd;
        int b0 = (int)floor(p);
        double val = 0.0;
        for (int b = b0; b <= b0 + 1; ++b)
            if (b >= 0 && b < nd) val += hat_weight(p - (double)b, a) * gz[(int64_t)k * nd + b];
        for (int j = 0; j < m; ++j) acc[j] += P->phi[(int64_t)j * na + k] * val;
    }
}

void cp4d_ref_adjoint(const ref_prob *P, const double *g, double *f) {
    const int n = P->n, m = P->m, na = P->n_angles, nd = P->nd;
    const int64_t nvox = (int64_t)P->nz * n * n;
#pragma omp parallel for schedule(dynamic, 256) num_threads(g_threads)
    for (int64_t v = 0; v < nvox; ++v) {
        int z = (int)(v / ((int64_t)n * n)), iy = (int)((v / n) % n), ix = (int)(v % n);
        double acc[64];
        for (int j = 0; j < m; ++j) acc[j] = 0.0;
        adjoint_voxel(P, g + (int64_t)z * na * nd, iy, ix, 0, na, acc);
        for (int j = 0; j < m; ++j) f[v * m + j] = acc[j];
    }
}

/* A8 adjoint with folding: gt_j[i,b] = sum_q phi[j,q n0+i] g[q n0+i, flip_q b],
 * then one backprojection over the base angles [0,pi). */
void cp4d_ref_adjoint_folded(const ref_prob *P, const double *g, double *f) {
    const int n = P->n, m = P->m, na = P->n_angles, nd = P->nd, n0 = na / P->n_half_rot;
    const int64_t nvox = (int64_t)P->nz * n * n;
    double *gt = (double *)calloc((size_t)P->nz * n0 * nd * m, sizeof(double)); /* [z][i][b][j] */
#pragma omp parallel for schedule(static) num_threads(g_threads)
    for (int64_t zi = 0; zi < (int64_t)P->nz * n0; ++zi) {
        int z = (int)(zi / n0), i = (int)(zi % n0);
        for (int b = 0; b < nd; ++b)
            for (int q = 0; q < P->n_half_rot; ++q) {
                int k = q * n0 + i, bb = (q & 1) ? nd - 1 - b : b;
                double gv = g[((int64_t)z * na + k) * nd + bb];
                for (int j = 0; j < m; ++j) gt[(zi * nd + b) * m + j] += P->phi[(int64_t)j * na + k] * gv;
            }
    }
    const double cen = 0.5 * (n - 1), cd = 0.5 * (nd - 1);
#pragma omp parallel for schedule(dynamic, 256) num_threads(g_threads)
    for (int64_t v = 0; v < nvox; ++v) {
        int z = (int)(v / ((int64_t)n * n)), iy = (int)((v / n) % n), ix = (int)(v % n);
        double acc[64], x = ix - cen, y = iy - cen;
        for (int j = 0; j < m; ++j) acc[j] = 0.0;
        for (int i = 0; i < n0; ++i) {
            double th = theta_of(P, i), c = cos(th), s = sin(th), a = fmax(fabs(c), fabs(s));
            double p = x * c + y * s + cd;
            int b0 = (int)floor(p);
            for (int b = b0; b <= b0 + 1; ++b)
                if (b >= 0 && b < nd) {
                    double w = hat_weight(p - (double)b, a);
                    const double *row = gt + (((int64_t)z * n0 + i) * nd + b) * m;
                    for (int j = 0; j < m; ++j) acc[j] += w * row[j];
                }
        }
        for (int j = 0; j < m; ++j) f[v * m + j] = acc[j];
    }
    free(gt);
}

/* adjoint at sampled voxels (z,iy,ix): out[i*m + j]; O(n_angles*m) each */
void cp4d_ref_adjoint_voxels(const ref_prob *P, const double *g, int64_t ns, const int32_t *zyx, double *out) {
    const int m = P->m;
#pragma omp parallel for schedule(dynamic, 16) num_threads(g_threads)
    for (int64_t i = 0; i < ns; ++i) {
        double acc[64];
        for (int j = 0; j < m; ++j) acc[j] = 0.0;
        adjoint_voxel(P, g + (int64_t)zyx[3 * i] * P->n_angles * P->nd, zyx[3 * i + 1], zyx[3 * i + 2], 0,
                      P->n_angles, acc);
        for (int j = 0; j < m; ++j) out[i * m + j] = acc[j];
    }
}

/* dense row of the static system matrix for angle index k (closed form), for the brute-force pins:
 * A[b][iy*n+ix], size nd x n*n */
void cp4d_ref_dense_A(const ref_prob *P, int k, double *A) {
    const int n = P->n, nd = P->nd;
    double th = theta_of(P, k), c = cos(th), s = sin(th), a = fmax(fabs(c), fabs(s));
    for (int b = 0; b < nd; ++b)
        for (int iy = 0; iy < n; ++iy)
            for (int ix = 0; ix < n; ++ix) {
                double u = (ix - 0.5 * (n - 1)) * c + (iy - 0.5 * (n - 1)) * s - (b - 0.5 * (nd - 1));
                A[((int64_t)b * n + iy) * n + ix] = hat_weight(u, a);
            }
}

/* ---------------------------------------------------------------------------------------------
 * O4  gradient / divergence (reading R4; Eq. 5).
 * Axes a = x, y, z, t (t = the 4th, coefficient axis of length m), weights w = (1,1,1,lambda2).
 * (d_a f)[i] = w_a (f[i+1]-f[i]) for i < n_a-1, 0 at i = n_a-1.   div p = -sum_a d_a^T p_a.
 * ------------------------------------------------------------------------------------------- */
static inline void axis_info(const ref_prob *P, int a, int *len, int64_t *stride) {
    const int64_t m = P->m, n = P->n;
    switch (a) {
    case 0: *len = P->n; *stride = m; break;
    case 1: *len = P->n; *stride = m * n; break;
    case 2: *len = P->nz; *stride = m * n * n; break;
    default: *len = P->m; *stride = 1; break;
    }
}
static inline int coord_of(const ref_prob *P, int64_t e, int a) {
    const int64_t m = P->m, n = P->n;
    switch (a) {
    case 0: return (int)((e / m) % n);
    case 1: return (int)((e / (m * n)) % n);
    case 2: return (int)(e / (m * n * n));
    default: return (int)(e % m);
    }
}

void cp4d_ref_grad(const ref_prob *P, const double *f, double *p) {
    const int64_t V = V_of(P);
    for (int a = 0; a < 4; ++a) {
        int len; int64_t st; axis_info(P, a, &len, &st);
        double w = (a == 3) ? P->lambda2 : 1.0;
#pragma omp parallel for schedule(static) num_threads(g_threads)
        for (int64_t e = 0; e < V; ++e) {
            int i = coord_of(P, e, a);
            p[a * V + e] = (i < len - 1) ? w * (f[e + st] - f[e]) : 0.0;
        }
    }
}

void cp4d_ref_div(const ref_prob *P, const double *p, double *f) {
    const int64_t V = V_of(P);
#pragma omp parallel for schedule(static) num_threads(g_threads)
    for (int64_t e = 0; e < V; ++e) {
        double d = 0.0;
        for (int a = 0; a < 4; ++a) {
            int len; int64_t st; axis_info(P, a, &len, &st);
            if (len == 1) continue;
            double w = (a == 3) ? P->lambda2 : 1.0;
            int i = coord_of(P, e, a);
            const double *pa = p + a * V;
            if (i == 0) d += w * pa[e];
            else if (i < len - 1) d += w * (pa[e] - pa[e - st]);
            else d += -w * pa[e - st];
        }
        f[e] = d;
    }
}

/* O5  prox of sigma F1*:  (h + sigma (K1 ft - g)) / (1 + sigma).
 * kf = K1 ft is passed in. */
void cp4d_ref_prox_f1(int64_t S, double sigma, const double *kf, const double *g, double *h1) {
    for (int64_t i = 0; i < S; ++i) h1[i] = (h1[i] + sigma * (kf[i] - g[i])) / (1.0 + sigma);
}

/* O6  prox of sigma F2* (reading R5): pointwise projection of the 4-vector
 * q = h2 + sigma grad ft onto the ball of radius lambda1: q / max(1, |q|_2 / lambda1).
 * lambda1 = 0 is the special case h2 = 0 (P7(i)).  gr = grad ft is passed in. Returns #clamped. */
int64_t cp4d_ref_prox_f2(int64_t V, double sigma, double lambda1, const double *gr, double *h2) {
    int64_t clamped = 0;
    for (int64_t e = 0; e < V; ++e) {
        double q[4], nn = 0.0;
        for (int a = 0; a < 4; ++a) { q[a] = h2[a * V + e] + sigma * gr[a * V + e]; nn += q[a] * q[a]; }
        nn = sqrt(nn);
        if (lambda1 <= 0.0) { for (int a = 0; a < 4; ++a) h2[a * V + e] = 0.0; continue; }
        double den = nn / lambda1;
        if (den > 1.0) ++clamped; else den = 1.0;
        for (int a = 0; a < 4; ++a) h2[a * V + e] = q[a] / den;
    }
    return clamped;
}

/* ---------------------------------------------------------------------------------------------
 * O7  n_iters iterations of Fig. 2 on the state (f, ft, h1, h2), in place:
 *   3: h1 <- (h1 + sigma K1 ft - sigma g)/(1+sigma)
 *   4: h2 <- (h2 + sigma grad ft)/max(1, |h2 + sigma grad ft|/lambda1)
 *   5: f+ <- f - tau K1^T h1 + tau div h2
 *   6: ft <- f+ + theta (f+ - f)
 * folded != 0 uses the pi-folded operators (same results to rounding; pinned by P4).
 * ------------------------------------------------------------------------------------------- */
int64_t cp4d_ref_cp(const ref_prob *P, const double *g, double tau, double sigma, double theta, int n_iters,
                    int folded, double *f, double *ft, double *h1, double *h2) {
    const int64_t V = V_of(P), S = S_of(P);
    double *kf = (double *)malloc(sizeof(double) * (size_t)S);
    double *gr = (double *)malloc(sizeof(double) * (size_t)V * 4);
    double *bp = (double *)malloc(sizeof(double) * (size_t)V);
    double *dv = (double *)malloc(sizeof(double) * (size_t)V);
    int64_t clamped = 0;
    for (int it = 0; it < n_iters; ++it) {
        if (folded) cp4d_ref_forward_folded(P, ft, kf); else cp4d_ref_forward(P, ft, kf);
        cp4d_ref_prox_f1(S, sigma, kf, g, h1);
        cp4d_ref_grad(P, ft, gr);
        clamped = cp4d_ref_prox_f2(V, sigma, P->lambda1, gr, h2);
        if (folded) cp4d_ref_adjoint_folded(P, h1, bp); else cp4d_ref_adjoint(P, h1, bp);
        cp4d_ref_div(P, h2, dv);
        for (int64_t e = 0; e < V; ++e) {
            double fn = f[e] - tau * bp[e] + tau * dv[e];
            ft[e] = fn + theta * (fn - f[e]);
            f[e] = fn;
        }
    }
    free(kf); free(gr); free(bp); free(dv);
    return clamped;
}

/* O8  power iteration for L = ||K||, K = (K1; K2) (reading R8):
 *   y = K1^T K1 x - div(grad x),  L = sqrt(|y|/|x|),  x <- y/|y|.   x is overwritten.
 * use_k1 / use_k2 select the blocks (K2 alone is pinned against a closed form). */
double cp4d_ref_power(const ref_prob *P, double *x, int n_steps, int use_k1, int use_k2, int folded) {
    const int64_t V = V_of(P), S = S_of(P);
    double *kf = (double *)malloc(sizeof(double) * (size_t)S);
    double *gr = (double *)malloc(sizeof(double) * (size_t)V * 4);
    double *y = (double *)calloc((size_t)V, sizeof(double));
    double *d = (double *)malloc(sizeof(double) * (size_t)V);
    double L = 0.0, nx = 0.0;
    for (int64_t e = 0; e < V; ++e) nx += x[e] * x[e];
    nx = sqrt(nx);
    for (int64_t e = 0; e < V; ++e) x[e] /= nx;
    for (int it = 0; it < n_steps; ++it) {
        memset(y, 0, sizeof(double) * (size_t)V);
        if (use_k1) {
            if (folded) { cp4d_ref_forward_folded(P, x, kf); cp4d_ref_adjoint_folded(P, kf, y); }
            else { cp4d_ref_forward(P, x, kf); cp4d_ref_adjoint(P, kf, y); }
        }
        if (use_k2) {
            cp4d_ref_grad(P, x, gr);
            cp4d_ref_div(P, gr, d);
            for (int64_t e = 0; e < V; ++e) y[e] -= d[e];
        }
        double ny = 0.0;
        for (int64_t e = 0; e < V; ++e) ny += y[e] * y[e];
        ny = sqrt(ny);
        L = sqrt(ny); /* |x| = 1 */
        if (ny == 0.0) break;
        for (int64_t e = 0; e < V; ++e) x[e] = y[e] / ny;
    }
    free(kf); free(gr); free(y); free(d);
    return L;
}
