/* oracle/ora.c — CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct fp64 implementation of the spatial part of the tensor-tomography
 * forward model of arxiv 2504.16446 and of its exact transpose:
 *
 *   A0  geometry: Table I vectors, R_s = R_beta(beta_s) R_alpha(alpha_s)
 *       ray / voxel relation from Eq. 4
 *   A1  John transform P_{sjk,xyz} (Eq. 5) by Joseph's method with bilinear
 *       interpolation of the field
 *   A2  its exact transpose, written twice: scatter (the forward loops run
 *       backwards) and gather (per voxel)                                         DESIGN.md reading S9
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this.
 * It shares no code, header, table or helper with the CUDA library (paper_2504_16446_b200/csrc).
 * Inputs: volume float32 (the same bytes the GPU gets); everything else and all arithmetic in double.
 * The basis matrix (Eq. 3), basis maps (Eq. 6), loss and gradient (Eq. 9, 13) live in oracle/oracle.py.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Table I values at alpha=beta=0; axis-aligned
 * projections are exact axis sums; uniform cube closed form; ball chord lengths to O(1/n); dense
 * Lambda*Lambda matrix brute force on tiny volumes; 90-degree covariance; tilt-0 slice decoupling;
 * <Ax,y> = <x,A^T y>; scatter == gather == dense transpose.  Nothing here is "parity unpinned".
 *
 * Readings of the paper: S4 voxel/pixel centres at integers, rotation centre
 * (n-1)/2; S7 P includes the Joseph step a/|d_m|; S8 major axis = lowest index i with
 * |d_i| >= max|d| - 1e-6, every slab weight 1, zero outside the volume, no interpolation along m.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int shape[3];          /* X, Y, Z */
    int J, Kd, P;
    double a, b;           /* voxel size, pixel size (Eq. 4) */
    double *d;             /* [P][3] beam direction in sample frame, R_s^T p */
    double *js, *ks;       /* [P][3] detector axes in sample frame */
    double *joff, *koff;   /* [P] */
    int *m;                /* [P] major axis */
    double *w;             /* [P] Joseph step a/|d_m| */
} ora_geom;

/* right-handed rotation by theta about unit axis n (Rodrigues), row-major 3x3 */
static void rodrigues(const double n[3], double theta, double R[9])
{
    double c = cos(theta), s = sin(theta), t = 1.0 - c;
    R[0] = c + t * n[0] * n[0];        R[1] = t * n[0] * n[1] - s * n[2]; R[2] = t * n[0] * n[2] + s * n[1];
    R[3] = t * n[1] * n[0] + s * n[2]; R[4] = c + t * n[1] * n[1];        R[5] = t * n[1] * n[2] - s * n[0];
    R[6] = t * n[2] * n[0] - s * n[1]; R[7] = t * n[2] * n[1] + s * n[0]; R[8] = c + t * n[2] * n[2];
}

static void matmul3(const double A[9], const double B[9], double C[9])
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            double s = 0;
            for (int k = 0; k < 3; k++) s += A[3 * i + k] * B[3 * k + j];
            C[3 * i + j] = s;
        }
}

/* out = R^T v */
static void matTvec(const double R[9], const double v[3], double out[3])
{
    for (int i = 0; i < 3; i++) out[i] = R[0 + i] * v[0] + R[3 + i] * v[1] + R[6 + i] * v[2];
}

/* vecs: p, j, k, inner_axis(alpha), outer_axis(beta), 3 doubles each (Table I) */
ora_geom *ora_geom_create(int X, int Y, int Z, int J, int Kd, int P, const double *rot, const double *tilt,
                          const double *joff, const double *koff, const double *vecs, double a, double b)
{
    ora_geom *g = (ora_geom *)calloc(1, sizeof(ora_geom));
    g->shape[0] = X; g->shape[1] = Y; g->shape[2] = Z;
    g->J = J; g->Kd = Kd; g->P = P; g->a = a; g->b = b;
    g->d = (double *)malloc(sizeof(double) * 3 * P);
    g->js = (double *)malloc(sizeof(double) * 3 * P);
    g->ks = (double *)malloc(sizeof(double) * 3 * P);
    g->joff = (double *)malloc(sizeof(double) * P);
    g->koff = (double *)malloc(sizeof(double) * P);
    g->w = (double *)malloc(sizeof(double) * P);
    g->m = (int *)malloc(sizeof(int) * P);
    for (int s = 0; s < P; s++) {
        double Ra[9], Rb[9], R[9];
        rodrigues(vecs + 9, rot[s], Ra);       /* inner "rotation" alpha about alpha-hat */
        rodrigues(vecs + 12, tilt[s], Rb);     /* outer "tilt" beta about beta-hat */
        matmul3(Rb, Ra, R);                    /* R_s = R_beta R_alpha */
        matTvec(R, vecs + 0, g->d + 3 * s);    /* sample-frame vectors R_s^T v */
        matTvec(R, vecs + 3, g->js + 3 * s);
        matTvec(R, vecs + 6, g->ks + 3 * s);
        g->joff[s] = joff ? joff[s] : 0.0;
        g->koff[s] = koff ? koff[s] : 0.0;
        const double *d = g->d + 3 * s;
        double mx = fmax(fabs(d[0]), fmax(fabs(d[1]), fabs(d[2])));
        int m = 0;
        while (fabs(d[m]) < mx - 1e-6) m++;    /* reading S8: lowest index within 1e-6 of the max */
        g->m[s] = m;
        g->w[s] = a / fabs(d[m]);              /* reading S7: path length per slab */
    }
    return g;
}

void ora_geom_destroy(ora_geom *g)
{
    if (!g) return;
    free(g->d); free(g->js); free(g->ks); free(g->joff); free(g->koff); free(g->w); free(g->m); free(g);
}

void ora_geom_get(const ora_geom *g, int s, double d[3], double js[3], double ks[3], int *m, double *w)
{
    memcpy(d, g->d + 3 * s, 24); memcpy(js, g->js + 3 * s, 24); memcpy(ks, g->ks + 3 * s, 24);
    *m = g->m[s]; *w = g->w[s];
}

/* point o on ray (j,k) of projection s with zero component along d: x(t) = o + t d.
 * From Eq. 4 a voxel at x lies on the ray iff (a/b) js.(x-xc) = j - jc - dj  (same for k), so the ray
 * sits at tau_j = (b/a)(j - jc - dj), tau_k likewise, in voxel units from the volume centre. */
static void ray_origin(const ora_geom *g, int s, int j, int k, double o[3])
{
    double tj = (g->b / g->a) * ((double)j - 0.5 * (g->J - 1) - g->joff[s]);
    double tk = (g->b / g->a) * ((double)k - 0.5 * (g->Kd - 1) - g->koff[s]);
    for (int i = 0; i < 3; i++)
        o[i] = 0.5 * (g->shape[i] - 1) + tj * g->js[3 * s + i] + tk * g->ks[3 * s + i];
}

/* in-slab position (pu,pv) of the ray at slab n of the major axis */
static void ray_at_slab(const ora_geom *g, int s, const double o[3], int n, int u, int v, double *pu, double *pv)
{
    const double *d = g->d + 3 * s;
    int m = g->m[s];
    double t = ((double)n - o[m]) / d[m];
    *pu = o[u] + t * d[u];
    *pv = o[v] + t * d[v];
}

static inline size_t vox_index(const ora_geom *g, int m, int u, int v, int n, int xu, int xv)
{
    int x[3];
    x[m] = n; x[u] = xu; x[v] = xv;
    return ((size_t)x[0] * g->shape[1] + x[1]) * g->shape[2] + x[2];
}

static void axes_uv(int m, int *u, int *v)
{
    *u = (m == 0) ? 1 : 0;
    *v = (m == 2) ? 1 : 2;
}

/* A1: one ray.  acc[K] (double) = w_s * sum over slabs of the bilinear interpolation of the field. */
static void joseph_ray(const ora_geom *g, const float *vol, int K, int ldk, int s, int j, int k, double *acc)
{
    int m = g->m[s], u, v;
    axes_uv(m, &u, &v);
    double o[3];
    ray_origin(g, s, j, k, o);
    for (int i = 0; i < K; i++) acc[i] = 0.0;
    for (int n = 0; n < g->shape[m]; n++) {
        double pu, pv;
        ray_at_slab(g, s, o, n, u, v, &pu, &pv);
        double fl_u = floor(pu), fl_v = floor(pv);
        int iu = (int)fl_u, iv = (int)fl_v;
        double fu = pu - fl_u, fv = pv - fl_v;
        for (int da = 0; da < 2; da++)
            for (int db = 0; db < 2; db++) {
                int xu = iu + da, xv = iv + db;
                if (xu < 0 || xu >= g->shape[u] || xv < 0 || xv >= g->shape[v]) continue;   /* zero outside */
                double wgt = (da ? fu : 1.0 - fu) * (db ? fv : 1.0 - fv);
                const float *c = vol + vox_index(g, m, u, v, n, xu, xv) * (size_t)ldk;
                for (int i = 0; i < K; i++) acc[i] += wgt * (double)c[i];
            }
    }
    for (int i = 0; i < K; i++) acc[i] *= g->w[s];
}

/* proj[(s-s0)][J][Kd][K] for projections s0 <= s < s1 */
void ora_john_forward(const ora_geom *g, const float *vol, int K, int ldk, int s0, int s1, double *proj,
                      int nthreads)
{
    long nray = (long)(s1 - s0) * g->J * g->Kd;
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads)
    for (long r = 0; r < nray; r++) {
        int k = (int)(r % g->Kd), j = (int)((r / g->Kd) % g->J), s = s0 + (int)(r / ((long)g->Kd * g->J));
        joseph_ray(g, vol, K, ldk, s, j, k, proj + (size_t)r * K);
    }
}

/* sampled rays: sjk[nray][3] -> out[nray][K] */
void ora_john_forward_rays(const ora_geom *g, const float *vol, int K, int ldk, long nray, const int32_t *sjk,
                           double *out, int nthreads)
{
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
    for (long r = 0; r < nray; r++)
        joseph_ray(g, vol, K, ldk, sjk[3 * r], sjk[3 * r + 1], sjk[3 * r + 2], out + (size_t)r * K);
}

/* A2 (i) scatter: the loops of joseph_ray with the assignment reversed.  y[P][J][Kd][K] -> out[X][Y][Z][K]
 * (out is zeroed here).  Single-threaded: scattered additions collide. */
void ora_john_adjoint_scatter(const ora_geom *g, const double *y, int K, double *out)
{
    size_t nvox = (size_t)g->shape[0] * g->shape[1] * g->shape[2];
    memset(out, 0, sizeof(double) * nvox * K);
    for (int s = 0; s < g->P; s++) {
        int m = g->m[s], u, v;
        axes_uv(m, &u, &v);
        for (int j = 0; j < g->J; j++)
            for (int k = 0; k < g->Kd; k++) {
                const double *yy = y + (((size_t)s * g->J + j) * g->Kd + k) * K;
                double o[3];
                ray_origin(g, s, j, k, o);
                for (int n = 0; n < g->shape[m]; n++) {
                    double pu, pv;
                    ray_at_slab(g, s, o, n, u, v, &pu, &pv);
                    double fl_u = floor(pu), fl_v = floor(pv);
                    int iu = (int)fl_u, iv = (int)fl_v;
                    double fu = pu - fl_u, fv = pv - fl_v;
                    for (int da = 0; da < 2; da++)
                        for (int db = 0; db < 2; db++) {
                            int xu = iu + da, xv = iv + db;
                            if (xu < 0 || xu >= g->shape[u] || xv < 0 || xv >= g->shape[v]) continue;
                            double wgt = g->w[s] * (da ? fu : 1.0 - fu) * (db ? fv : 1.0 - fv);
                            double *c = out + vox_index(g, m, u, v, n, xu, xv) * (size_t)K;
                            for (int i = 0; i < K; i++) c[i] += wgt * yy[i];
                        }
                }
            }
    }
}

static double tri(double t) { t = fabs(t); return t < 1.0 ? 1.0 - t : 0.0; }

/* A2 (ii) gather, one voxel, projections s0..s1-1: every ray (jj,kk) that can come within one voxel of x in
 * the slab n = x[m] is re-traced exactly as in the forward, and weighted by
 * Lambda(pu - x_u) Lambda(pv - x_v) = the bilinear weight the forward gave that voxel.
 * If taps != NULL, the visited (s,jj,kk,weight) with weight > 0 are appended instead of accumulating. */
static long gather_voxel(const ora_geom *g, const double *y, int K, int x0, int x1, int x2, int s0, int s1,
                         double *acc, double *taps, long maxtaps)
{
    int x[3] = {x0, x1, x2};
    long ntaps = 0;
    for (int s = s0; s < s1; s++) {
        int m = g->m[s], u, v;
        axes_uv(m, &u, &v);
        const double *js = g->js + 3 * s, *ks = g->ks + 3 * s;
        double rel[3];
        for (int i = 0; i < 3; i++) rel[i] = (double)x[i] - 0.5 * (g->shape[i] - 1);
        double ab = g->a / g->b;
        double j0 = 0.5 * (g->J - 1) + g->joff[s] + ab * (js[0] * rel[0] + js[1] * rel[1] + js[2] * rel[2]);
        double k0 = 0.5 * (g->Kd - 1) + g->koff[s] + ab * (ks[0] * rel[0] + ks[1] * rel[1] + ks[2] * rel[2]);
        /* a ray within one voxel (in u and v) of x lands within ab*(|js_u|+|js_v|) of j0; search a
         * window one pixel wider than that */
        int rj = (int)ceil(ab * (fabs(js[u]) + fabs(js[v]))) + 1;
        int rk = (int)ceil(ab * (fabs(ks[u]) + fabs(ks[v]))) + 1;
        for (int jj = (int)floor(j0) - rj; jj <= (int)floor(j0) + rj + 1; jj++)
            for (int kk = (int)floor(k0) - rk; kk <= (int)floor(k0) + rk + 1; kk++) {
                if (jj < 0 || jj >= g->J || kk < 0 || kk >= g->Kd) continue;   /* no such ray */
                double o[3], pu, pv;
                ray_origin(g, s, jj, kk, o);
                ray_at_slab(g, s, o, x[m], u, v, &pu, &pv);
                double wgt = g->w[s] * tri(pu - x[u]) * tri(pv - x[v]);
                if (wgt <= 0.0) continue;
                if (taps) {
                    if (ntaps < maxtaps) {
                        taps[4 * ntaps + 0] = s; taps[4 * ntaps + 1] = jj;
                        taps[4 * ntaps + 2] = kk; taps[4 * ntaps + 3] = wgt;
                    }
                    ntaps++;
                } else {
                    const double *yy = y + (((size_t)s * g->J + jj) * g->Kd + kk) * K;
                    for (int i = 0; i < K; i++) acc[i] += wgt * yy[i];
                }
            }
    }
    return ntaps;
}

void ora_john_adjoint_gather(const ora_geom *g, const double *y, int K, double *out, int nthreads)
{
    long nvox = (long)g->shape[0] * g->shape[1] * g->shape[2];
#pragma omp parallel for schedule(dynamic, 256) num_threads(nthreads)
    for (long q = 0; q < nvox; q++) {
        int z = (int)(q % g->shape[2]), yy = (int)((q / g->shape[2]) % g->shape[1]);
        int x = (int)(q / ((long)g->shape[2] * g->shape[1]));
        double *acc = out + (size_t)q * K;
        for (int i = 0; i < K; i++) acc[i] = 0.0;
        gather_voxel(g, y, K, x, yy, z, 0, g->P, acc, NULL, 0);
    }
}

/* sampled voxels xyz[nvox][3] -> out[nvox][K] */
void ora_john_adjoint_voxels(const ora_geom *g, const double *y, int K, long nvox, const int32_t *xyz,
                             double *out, int nthreads)
{
#pragma omp parallel for schedule(dynamic, 4) num_threads(nthreads)
    for (long q = 0; q < nvox; q++) {
        double *acc = out + (size_t)q * K;
        for (int i = 0; i < K; i++) acc[i] = 0.0;
        gather_voxel(g, y, K, xyz[3 * q], xyz[3 * q + 1], xyz[3 * q + 2], 0, g->P, acc, NULL, 0);
    }
}

/* rows (s, jj, kk, P_{s jj kk, xyz}) of the non-zero column entries of voxel (x0,x1,x2); returns the count
 * (may exceed maxtaps, in which case only maxtaps rows were written) */
long ora_voxel_taps(const ora_geom *g, int x0, int x1, int x2, double *taps, long maxtaps)
{
    return gather_voxel(g, NULL, 0, x0, x1, x2, 0, g->P, NULL, taps, maxtaps);
}

/* dense P_s for brute-force pins on tiny problems: mat[J*Kd][X*Y*Z] from the closed form
 * P = w_s Lambda(pu(j,k;n=x_m) - x_u) Lambda(pv - x_v)  (A1) — no floor(), no tap loop. */
void ora_dense_matrix(const ora_geom *g, int s, double *mat)
{
    int m = g->m[s], u, v;
    axes_uv(m, &u, &v);
    size_t nvox = (size_t)g->shape[0] * g->shape[1] * g->shape[2];
    for (int j = 0; j < g->J; j++)
        for (int k = 0; k < g->Kd; k++) {
            double o[3];
            ray_origin(g, s, j, k, o);
            double *row = mat + ((size_t)j * g->Kd + k) * nvox;
            for (int x0 = 0; x0 < g->shape[0]; x0++)
                for (int x1 = 0; x1 < g->shape[1]; x1++)
                    for (int x2 = 0; x2 < g->shape[2]; x2++) {
                        int x[3] = {x0, x1, x2};
                        double pu, pv;
                        ray_at_slab(g, s, o, x[m], u, v, &pu, &pv);
                        row[((size_t)x0 * g->shape[1] + x1) * g->shape[2] + x2] =
                            g->w[s] * tri(pu - x[u]) * tri(pv - x[v]);
                    }
        }
}

/* NEXT-1 (reading S9, second half): the adjoint AS THE PAPER DESCRIBES IT, PAPER.md:314 — "bilinear
 * interpolation ... of the projection for the adjoint".  Voxel-driven and NOT the transpose of joseph_ray: for each
 * voxel x and projection s the detector position (j0,k0) of the voxel follows from Eq. 4,
 *     j0 = jc + dj_s + (a/b) js.(x - xc),   k0 = kc + dk_s + (a/b) ks.(x - xc),
 * the projection is interpolated bilinearly at (j0,k0) (pixels outside the detector count as 0) and the value
 * is weighted by the same Joseph step w_s = a/|d_m| the forward uses, so both operators carry path-length units:
 *     out[x][i] = sum_s w_s sum_{a,b in {0,1}} (a ? fj : 1-fj)(b ? fk : 1-fk) y[s][jb+a][kb+b][i].
 * y[P][J][Kd][K] -> out[X][Y][Z][K].  Pins: tests/test_oracle_backproject.py. */
static void backproject_voxel(const ora_geom *g, const double *y, int K, const int x[3], double *acc)
{
    double ab = g->a / g->b;
    for (int i = 0; i < K; i++) acc[i] = 0.0;
    for (int s = 0; s < g->P; s++) {
        const double *js = g->js + 3 * s, *ks = g->ks + 3 * s;
        double j0 = 0.5 * (g->J - 1) + g->joff[s], k0 = 0.5 * (g->Kd - 1) + g->koff[s];
        for (int i = 0; i < 3; i++) {
            double rel = (double)x[i] - 0.5 * (g->shape[i] - 1);
            j0 += ab * js[i] * rel; k0 += ab * ks[i] * rel;
        }
        double flj = floor(j0), flk = floor(k0);
        int jb = (int)flj, kb = (int)flk;
        double fj = j0 - flj, fk = k0 - flk;
        for (int da = 0; da < 2; da++)
            for (int db = 0; db < 2; db++) {
                int jj = jb + da, kk = kb + db;
                if (jj < 0 || jj >= g->J || kk < 0 || kk >= g->Kd) continue;      /* no such pixel */
                double wgt = g->w[s] * (da ? fj : 1.0 - fj) * (db ? fk : 1.0 - fk);
                const double *yy = y + (((size_t)s * g->J + jj) * g->Kd + kk) * K;
                for (int i = 0; i < K; i++) acc[i] += wgt * yy[i];
            }
    }
}

void ora_john_backproject_bilinear(const ora_geom *g, const double *y, int K, double *out, int nthreads)
{
    long nvox = (long)g->shape[0] * g->shape[1] * g->shape[2];
#pragma omp parallel for schedule(dynamic, 256) num_threads(nthreads)
    for (long q = 0; q < nvox; q++) {
        int x[3];
        x[2] = (int)(q % g->shape[2]); x[1] = (int)((q / g->shape[2]) % g->shape[1]);
        x[0] = (int)(q / ((long)g->shape[2] * g->shape[1]));
        backproject_voxel(g, y, K, x, out + (size_t)q * K);
    }
}

/* sampled voxels xyz[nvox][3] -> out[nvox][K] (full-size parity samples) */
void ora_john_backproject_bilinear_voxels(const ora_geom *g, const double *y, int K, long nvox, const int32_t *xyz,
                                          double *out)
{
    for (long q = 0; q < nvox; q++) {
        int x[3] = {xyz[3 * q], xyz[3 * q + 1], xyz[3 * q + 2]};
        backproject_voxel(g, y, K, x, out + (size_t)q * K);
    }
}
