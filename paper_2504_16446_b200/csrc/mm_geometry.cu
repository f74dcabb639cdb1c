// mm_geometry.cu — host side of the library: geometry / ray setup (step a1) and the spherical-harmonic
// basis-matrix helper (step a2).  All fp64, runs once per geometry.  Citations: P:NN = PAPER.md line NN.
#include <cuda_runtime.h>
#include <math.h>
#include <algorithm>
#include <string.h>

#include <new>

#include "mm_internal.h"

static thread_local std::string g_last_error;

void mm_set_error(const std::string &msg) { g_last_error = msg; }

extern "C" const char *mm_last_error(void) { return g_last_error.c_str(); }

extern "C" const char *mm_status_string(mm_status s)
{
    switch (s) {
        case MM_OK: return "MM_OK";
        case MM_ERR_NULL: return "MM_ERR_NULL";
        case MM_ERR_SHAPE: return "MM_ERR_SHAPE";
        case MM_ERR_VALUE: return "MM_ERR_VALUE";
        case MM_ERR_ALLOC: return "MM_ERR_ALLOC";
        case MM_ERR_CUDA: return "MM_ERR_CUDA";
        case MM_ERR_UNSUPPORTED: return "MM_ERR_UNSUPPORTED";
    }
    return "MM_ERR_?";
}

namespace {

struct V3 {
    double x[3];
};

inline double dot3(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

// Right-handed rotation by angle t about unit axis n (reading S6), row-major.
void rotation_about(const double n[3], double t, double R[9])
{
    const double c = cos(t), s = sin(t), omc = 1.0 - c;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) R[3 * i + j] = omc * n[i] * n[j] + (i == j ? c : 0.0);
    R[1] -= s * n[2]; R[2] += s * n[1];
    R[3] += s * n[2]; R[5] -= s * n[0];
    R[6] -= s * n[1]; R[7] += s * n[0];
}

// take the user's direction, or the Table I standard when it is all-zero; must be unit length
bool pick_dir(const double in[3], double sx, double sy, double sz, double out[3])
{
    if (in[0] == 0.0 && in[1] == 0.0 && in[2] == 0.0) {
        out[0] = sx; out[1] = sy; out[2] = sz;
        return true;
    }
    for (int i = 0; i < 3; i++)
        if (!isfinite(in[i])) return false;
    const double n = sqrt(dot3(in, in));
    if (fabs(n - 1.0) > 1e-9) return false;
    for (int i = 0; i < 3; i++) out[i] = in[i] / n;
    return true;
}

}  // namespace

extern "C" mm_status mm_geometry_create(const mm_geometry_desc *desc, mm_geometry **out)
{
    if (!desc || !out) { mm_set_error("mm_geometry_create: NULL desc/out"); return MM_ERR_NULL; }
    *out = nullptr;
    if (!desc->rotations || !desc->tilts) { mm_set_error("mm_geometry_create: NULL rotations/tilts"); return MM_ERR_NULL; }
    for (int i = 0; i < 3; i++)
        if (desc->volume_shape[i] < 1 || desc->volume_shape[i] > 32768) { mm_set_error("volume_shape out of range"); return MM_ERR_SHAPE; }
    if (desc->det_shape[0] < 1 || desc->det_shape[1] < 1 || desc->det_shape[0] > 32768 || desc->det_shape[1] > 32768 ||
        desc->n_proj < 1) { mm_set_error("det_shape / n_proj out of range"); return MM_ERR_SHAPE; }
    double p[3], jd[3], kd[3], q0[3], q90[3], ia[3], oa[3];
    // Table I standard values (row 2 garbled: reading S1)
    if (!pick_dir(desc->p_dir, 0, 0, 1, p) || !pick_dir(desc->j_dir, 0, 1, 0, jd) || !pick_dir(desc->k_dir, 1, 0, 0, kd) ||
        !pick_dir(desc->q0_dir, 1, 0, 0, q0) || !pick_dir(desc->q90_dir, 0, 1, 0, q90) ||
        !pick_dir(desc->inner_axis, 0, 1, 0, ia) || !pick_dir(desc->outer_axis, 1, 0, 0, oa)) {
        mm_set_error("direction vectors must be finite and of unit length");
        return MM_ERR_VALUE;
    }
    if (fabs(dot3(p, jd)) > 1e-9 || fabs(dot3(p, kd)) > 1e-9 || fabs(dot3(jd, kd)) > 1e-9) {
        mm_set_error("p, j, k must be mutually orthogonal");
        return MM_ERR_VALUE;
    }
    const double a = desc->voxel_size == 0.0 ? 1.0 : desc->voxel_size;
    const double b = desc->pixel_size == 0.0 ? 1.0 : desc->pixel_size;
    if (!(a > 0.0) || !(b > 0.0) || !isfinite(a) || !isfinite(b)) { mm_set_error("voxel_size/pixel_size must be positive"); return MM_ERR_VALUE; }
    const int P = desc->n_proj;
    for (int s = 0; s < P; s++) {
        if (!isfinite(desc->rotations[s]) || !isfinite(desc->tilts[s]) ||
            (desc->j_offsets && !isfinite(desc->j_offsets[s])) || (desc->k_offsets && !isfinite(desc->k_offsets[s]))) {
            mm_set_error("non-finite angle or offset");
            return MM_ERR_VALUE;
        }
    }
    mm_geometry *g = new (std::nothrow) mm_geometry();
    if (!g) { mm_set_error("host allocation failed"); return MM_ERR_ALLOC; }
    for (int i = 0; i < 3; i++) g->shape[i] = desc->volume_shape[i];
    g->J = desc->det_shape[0]; g->Kd = desc->det_shape[1]; g->P = P; g->a = a; g->b = b;
    memcpy(g->q0, q0, sizeof q0); memcpy(g->q90, q90, sizeof q90); memcpy(g->p, p, sizeof p);
    g->d_table = nullptr;
    g->host.resize(P);
    g->table.resize(P);
    const double xc[3] = {0.5 * (g->shape[0] - 1), 0.5 * (g->shape[1] - 1), 0.5 * (g->shape[2] - 1)};   // S4
    const double jc = 0.5 * (g->J - 1), kc = 0.5 * (g->Kd - 1);
    const double ba = b / a, ab = a / b;
    for (int s = 0; s < P; s++) {
        MMProjHost &h = g->host[s];
        double Ra[9], Rb[9];
        rotation_about(ia, desc->rotations[s], Ra);
        rotation_about(oa, desc->tilts[s], Rb);
        for (int i = 0; i < 3; i++)                          // R_s = R_beta R_alpha
            for (int j = 0; j < 3; j++) h.R[3 * i + j] = Rb[3 * i] * Ra[j] + Rb[3 * i + 1] * Ra[3 + j] + Rb[3 * i + 2] * Ra[6 + j];
        for (int i = 0; i < 3; i++) {                        // sample-frame vectors R_s^T v
            h.d[i] = h.R[i] * p[0] + h.R[3 + i] * p[1] + h.R[6 + i] * p[2];
            h.js[i] = h.R[i] * jd[0] + h.R[3 + i] * jd[1] + h.R[6 + i] * jd[2];
            h.ks[i] = h.R[i] * kd[0] + h.R[3 + i] * kd[1] + h.R[6 + i] * kd[2];
        }
        const double big = fmax(fabs(h.d[0]), fmax(fabs(h.d[1]), fabs(h.d[2])));
        int m = 2;
        if (fabs(h.d[0]) >= big - 1e-6) m = 0;               // reading S8: lowest index within 1e-6 of the max
        else if (fabs(h.d[1]) >= big - 1e-6) m = 1;
        const int u = (m == 0) ? 1 : 0, v = (m == 2) ? 1 : 2;
        h.m = m;
        h.w = a / fabs(h.d[m]);                              // reading S7
        const double dj = desc->j_offsets ? desc->j_offsets[s] : 0.0, dk = desc->k_offsets ? desc->k_offsets[s] : 0.0;
        MMProj &t = g->table[s];
        t.m = m; t.u = u; t.v = v;
        t.w = (float)h.w;
        // ray (j,k): x(t) = xc + tau_j js + tau_k ks + t d, tau_j = (b/a)(j - jc - dj)   (Eq. 4 solved for the ray)
        // at slab n: t = (n - x_m(0))/d_m  =>  pu = x_u(0) + (n - x_m(0)) d_u/d_m
        t.su = h.d[u] / h.d[m];
        t.sv = h.d[v] / h.d[m];
        t.Mju = ba * (h.js[u] - t.su * h.js[m]);
        t.Mku = ba * (h.ks[u] - t.su * h.ks[m]);
        t.Mjv = ba * (h.js[v] - t.sv * h.js[m]);
        t.Mkv = ba * (h.ks[v] - t.sv * h.ks[m]);
        t.Cu = xc[u] - t.su * xc[m] - (jc + dj) * t.Mju - (kc + dk) * t.Mku;
        t.Cv = xc[v] - t.sv * xc[m] - (jc + dj) * t.Mjv - (kc + dk) * t.Mkv;
        t.su_fx = llrint(ldexp(t.su, 40));
        t.sv_fx = llrint(ldexp(t.sv, 40));
        t.w64 = h.w;
        // voxel -> detector: j0 = jc + dj + (a/b) js.(x - xc)
        t.Jc = jc + dj; t.Kc = kc + dk;
        for (int i = 0; i < 3; i++) {
            t.Jx[i] = ab * h.js[i]; t.Kx[i] = ab * h.ks[i];
            t.Jc -= t.Jx[i] * xc[i]; t.Kc -= t.Kx[i] * xc[i];
        }
        t.mju = (float)t.Mju; t.mku = (float)t.Mku; t.mjv = (float)t.Mjv; t.mkv = (float)t.Mkv;
        const double det = t.Mju * t.Mkv - t.Mku * t.Mjv;   // never 0: d_m != 0
        // (dj,dk) = M^-1 (du,dv), |du|,|dv| < 1  =>  |dj| < (|Mkv| + |Mku|)/|det|, |dk| < (|Mjv| + |Mju|)/|det|
        t.hj = (float)((fabs(t.Mkv) + fabs(t.Mku)) / fabs(det) * (1.0 + 1e-6) + 1e-6);
        t.hk = (float)((fabs(t.Mjv) + fabs(t.Mju)) / fabs(det) * (1.0 + 1e-6) + 1e-6);
        // half-width <= 1: at most 2 candidate rays along that detector axis; < 1.5: at most 3
        t.gcode = (t.hj < 1.5f && t.hk < 1.5f) ? 4 + 2 * (t.hj <= 1.000003f ? 0 : 1) + (t.hk <= 1.000003f ? 0 : 1) : 1;
        t.pad_ = 0;
    }
    // Detector tile of the brick adjoint (mm_adjoint_brick.cu): a 4 x 4 x 8 brick of voxels spans
    // ext = 3|Jx| + 3|Jy| + 7|Jz| pixels along j; with the tile origin two pixels below the nearest pixel of the lowest
    // corner and 3-wide candidate windows the indices used are 0 .. floor(ext + 3) + 1.
    g->brick_tj = g->brick_tk = 0;
    {
        int tj = 0, tk = 0;
        bool ok = true;
        for (int s = 0; s < P && ok; s++) {
            const MMProj &t = g->table[s];
            if (t.gcode < 4) { ok = false; break; }
            const double ej = 3.0 * fabs(t.Jx[0]) + 3.0 * fabs(t.Jx[1]) + 7.0 * fabs(t.Jx[2]);
            const double ek = 3.0 * fabs(t.Kx[0]) + 3.0 * fabs(t.Kx[1]) + 7.0 * fabs(t.Kx[2]);
            tj = std::max(tj, (int)floor(ej + 3.0 + 1e-3) + 2);
            tk = std::max(tk, (int)floor(ek + 3.0 + 1e-3) + 2);
        }
        tk |= 1;                                             // odd row pitch: rows start in different shared-memory banks
        if (ok && tj <= 16 && tk <= 17) { g->brick_tj = tj; g->brick_tk = tk; }
    }
    // Upload the table.  On a machine without a CUDA device the geometry stays host-only (mm_geometry_get and
    // mm_basis_sh_matrix work; every device call then fails with MM_ERR_CUDA — there is no CPU fallback).
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        g->device = -1;
        *out = g;
        return MM_OK;
    }
    if (cudaGetDevice(&g->device) != cudaSuccess) {
        mm_set_error(std::string("cudaGetDevice: ") + cudaGetErrorString(cudaGetLastError()));
        delete g;
        return MM_ERR_CUDA;
    }
    cudaError_t e = cudaMalloc((void **)&g->d_table, sizeof(MMProj) * (size_t)P);
    if (e != cudaSuccess) {
        mm_set_error(std::string("cudaMalloc(ray table): ") + cudaGetErrorString(e));
        cudaGetLastError();
        delete g;
        return MM_ERR_ALLOC;
    }
    e = cudaMemcpy(g->d_table, g->table.data(), sizeof(MMProj) * (size_t)P, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        mm_set_error(std::string("cudaMemcpy(ray table): ") + cudaGetErrorString(e));
        cudaFree(g->d_table);
        delete g;
        return MM_ERR_CUDA;
    }
    *out = g;
    return MM_OK;
}

extern "C" mm_status mm_geometry_destroy(mm_geometry *g)
{
    if (!g) return MM_OK;
    if (g->d_table) cudaFree(g->d_table);
    delete g;
    return MM_OK;
}

extern "C" mm_status mm_geometry_get(const mm_geometry *g, int32_t s, double d[3], double js[3], double ks[3],
                                     int32_t *major_axis, double *step)
{
    if (!g) { mm_set_error("mm_geometry_get: NULL geometry"); return MM_ERR_NULL; }
    if (s < 0 || s >= g->P) { mm_set_error("mm_geometry_get: projection index out of range"); return MM_ERR_SHAPE; }
    const MMProjHost &h = g->host[s];
    if (d) memcpy(d, h.d, sizeof h.d);
    if (js) memcpy(js, h.js, sizeof h.js);
    if (ks) memcpy(ks, h.ks, sizeof h.ks);
    if (major_axis) *major_axis = h.m;
    if (step) *step = h.w;
    return MM_OK;
}

// ------------------------------------------------------------------------------------------------
// Real spherical harmonics of even degree and the segment-averaged basis matrix, Eq. 3.
// ------------------------------------------------------------------------------------------------
namespace {

// Y[i] for even l <= L, i ordered l ascending then m = -l..l; 4pi-normalised (mean of Y^2 over the sphere
// is 1, Y_00 = 1), no Condon-Shortley phase; m < 0 carries sin(|m| phi), m > 0 carries cos(m phi) (S14).
// Uses Y_l,+-m = sqrt(2) N_lm T_lm(z) {Re,Im}(x+iy)^m with T_lm = d^m P_l / dz^m from the three-term recurrence.
void real_sh_even(int L, const double n[3], double *Y)
{
    const double x = n[0], y = n[1], z = n[2];
    double cre = 1.0, cim = 0.0;                 // (x + i y)^m
    double dfact = 1.0;                          // (2m-1)!!
    for (int m = 0; m <= L; m++) {
        if (m > 0) {
            const double nre = cre * x - cim * y, nim = cre * y + cim * x;
            cre = nre; cim = nim;
            dfact *= (2 * m - 1);
        }
        double t_lm2 = 0.0, t_lm1 = 0.0;
        for (int l = m; l <= L; l++) {
            double t;
            if (l == m) t = dfact;
            else if (l == m + 1) t = (2 * m + 1) * z * t_lm1;
            else t = ((2 * l - 1) * z * t_lm1 - (l + m - 1) * t_lm2) / (l - m);
            t_lm2 = t_lm1; t_lm1 = t;
            if (l & 1) continue;
            double ratio = 1.0;                  // (l-m)!/(l+m)!
            for (int q = l - m + 1; q <= l + m; q++) ratio /= q;
            const double N = sqrt((2 * l + 1) * ratio);
            const int base = l * (l - 1) / 2 + l;   // index of (l, 0): sum_{l'<l, even} (2l'+1) = l(l-1)/2
            if (m == 0) Y[base] = N * t;
            else {
                Y[base + m] = M_SQRT2 * N * t * cre;
                Y[base - m] = M_SQRT2 * N * t * cim;
            }
        }
    }
}

}  // namespace

static mm_status basis_sh_matrix(const mm_geometry *g, int32_t ell_max, double two_theta, int32_t D, const double *seg_start,
                                 const double *seg_end, float *h_B)
{
    if (!g || !seg_start || !seg_end || !h_B) { mm_set_error("mm_basis_sh_matrix: NULL argument"); return MM_ERR_NULL; }
    if (ell_max < 0 || (ell_max & 1) || ell_max > 64 || D < 1) { mm_set_error("ell_max must be even in [0,64], D >= 1"); return MM_ERR_SHAPE; }
    const int K = (ell_max + 1) * (ell_max + 2) / 2;
    // f_i(phi) = Y_i(R_s^T q(phi)) is a trigonometric polynomial of degree <= ell_max: sample it on
    // M > 2 ell_max equispaced angles, take its Fourier coefficients, integrate each harmonic in closed form.
    const int M = 2 * ell_max + 2;
    std::vector<double> samp((size_t)M * K), Y(K), ac((size_t)(ell_max + 1) * K), bc((size_t)(ell_max + 1) * K);
    const double ct = cos(0.5 * two_theta), st = sin(0.5 * two_theta);
    for (int s = 0; s < g->P; s++) {
        const double *R = g->host[s].R;
        for (int t = 0; t < M; t++) {
            const double phi = 2.0 * M_PI * t / M, c = cos(phi), sn = sin(phi);
            double q[3], qs[3];
            // Eq. 1: cos(theta)(cos phi q0 + sin phi q90) - sin(theta) p, theta = 2theta/2 (0: the small-angle line)
            for (int i = 0; i < 3; i++) q[i] = ct * (c * g->q0[i] + sn * g->q90[i]) - st * g->p[i];
            for (int i = 0; i < 3; i++) qs[i] = R[i] * q[0] + R[3 + i] * q[1] + R[6 + i] * q[2];   // R_s^T q
            real_sh_even(ell_max, qs, Y.data());
            for (int i = 0; i < K; i++) samp[(size_t)t * K + i] = Y[i];
        }
        for (int h = 0; h <= ell_max; h++)
            for (int i = 0; i < K; i++) {
                double sa = 0.0, sb = 0.0;
                for (int t = 0; t < M; t++) {
                    const double ang = 2.0 * M_PI * ((h * t) % M) / M;
                    sa += samp[(size_t)t * K + i] * cos(ang);
                    sb += samp[(size_t)t * K + i] * sin(ang);
                }
                const double sc = (h == 0) ? 1.0 / M : 2.0 / M;
                ac[(size_t)h * K + i] = sc * sa;
                bc[(size_t)h * K + i] = sc * sb;
            }
        for (int c = 0; c < D; c++) {
            const double p0 = seg_start[c], p1 = seg_end[c], wdt = p1 - p0;
            if (!isfinite(p0) || !isfinite(p1)) { mm_set_error("non-finite segment angle"); return MM_ERR_VALUE; }
            for (int i = 0; i < K; i++) {
                double val = ac[i];
                for (int h = 1; h <= ell_max; h++) {
                    double ca, sa;
                    if (fabs(wdt) > 1e-12) {
                        ca = (sin(h * p1) - sin(h * p0)) / (h * wdt);     // mean of cos(h phi)
                        sa = -(cos(h * p1) - cos(h * p0)) / (h * wdt);    // mean of sin(h phi)
                    } else {
                        ca = cos(h * p0); sa = sin(h * p0);
                    }
                    val += ac[(size_t)h * K + i] * ca + bc[(size_t)h * K + i] * sa;
                }
                h_B[((size_t)s * K + i) * D + c] = (float)val;
            }
        }
    }
    return MM_OK;
}

extern "C" mm_status mm_basis_sh_matrix(const mm_geometry *g, int32_t ell_max, int32_t D, const double *seg_start,
                                        const double *seg_end, float *h_B)
{
    return basis_sh_matrix(g, ell_max, 0.0, D, seg_start, seg_end, h_B);
}

extern "C" mm_status mm_basis_sh_matrix_2theta(const mm_geometry *g, int32_t ell_max, double two_theta, int32_t D,
                                               const double *seg_start, const double *seg_end, float *h_B)
{
    if (!isfinite(two_theta)) { mm_set_error("mm_basis_sh_matrix_2theta: non-finite 2theta"); return MM_ERR_VALUE; }
    return basis_sh_matrix(g, ell_max, two_theta, D, seg_start, seg_end, h_B);
}

// ------------------------------------------------------------------------------------------------
// NEXT-2: basis sets attached to a grid of orientations: nearest-neighbour indicators and
// Gaussian kernels.  Same Eq. 3 segment average, midpoint rule with n_quad points (reading S20).
// ------------------------------------------------------------------------------------------------
extern "C" mm_status mm_basis_grid_matrix(const mm_geometry *g, int32_t kind, int32_t n_dirs, const double *dirs, double sigma,
                                          int32_t D, const double *seg_start, const double *seg_end, int32_t n_quad, float *h_B)
{
    if (!g || !dirs || !seg_start || !seg_end || !h_B) { mm_set_error("mm_basis_grid_matrix: NULL argument"); return MM_ERR_NULL; }
    if (n_dirs < 1 || D < 1 || n_quad < 1) { mm_set_error("mm_basis_grid_matrix: need n_dirs, D, n_quad >= 1"); return MM_ERR_SHAPE; }
    if (kind != MM_BASIS_NN && kind != MM_BASIS_GK) { mm_set_error("mm_basis_grid_matrix: kind must be MM_BASIS_NN or MM_BASIS_GK"); return MM_ERR_VALUE; }
    if (kind == MM_BASIS_GK && !(sigma > 0.0)) { mm_set_error("mm_basis_grid_matrix: sigma must be positive"); return MM_ERR_VALUE; }
    std::vector<double> u((size_t)3 * n_dirs);                        // normalised grid directions
    for (int i = 0; i < n_dirs; i++) {
        const double *d = dirs + 3 * i;
        const double n = sqrt(dot3(d, d));
        if (!(n > 0.0) || !isfinite(n)) { mm_set_error("mm_basis_grid_matrix: zero or non-finite direction"); return MM_ERR_VALUE; }
        for (int a = 0; a < 3; a++) u[3 * i + a] = d[a] / n;
    }
    std::vector<double> acc(n_dirs);
    const double inv2s2 = kind == MM_BASIS_GK ? 0.5 / (sigma * sigma) : 0.0;
    for (int s = 0; s < g->P; s++) {
        const double *R = g->host[s].R;
        for (int c = 0; c < D; c++) {
            if (!isfinite(seg_start[c]) || !isfinite(seg_end[c])) { mm_set_error("non-finite segment angle"); return MM_ERR_VALUE; }
            for (int i = 0; i < n_dirs; i++) acc[i] = 0.0;
            for (int t = 0; t < n_quad; t++) {
                const double phi = seg_start[c] + (seg_end[c] - seg_start[c]) * ((t + 0.5) / n_quad);
                const double cp = cos(phi), sp = sin(phi);
                double q[3], qs[3];
                for (int a = 0; a < 3; a++) q[a] = cp * g->q0[a] + sp * g->q90[a];              // Eq. 1, small-angle line
                for (int a = 0; a < 3; a++) qs[a] = R[a] * q[0] + R[3 + a] * q[1] + R[6 + a] * q[2];   // R_s^T q
                if (kind == MM_BASIS_NN) {
                    int best = 0;
                    double bestc = -1.0;
                    for (int i = 0; i < n_dirs; i++) {
                        const double ca = fabs(dot3(qs, &u[3 * i]));
                        if (ca > bestc) { bestc = ca; best = i; }                                // first maximum wins ties
                    }
                    acc[best] += 1.0;
                } else {
                    for (int i = 0; i < n_dirs; i++) {
                        const double th = acos(fmin(fabs(dot3(qs, &u[3 * i])), 1.0));
                        acc[i] += exp(-th * th * inv2s2);
                    }
                }
            }
            for (int i = 0; i < n_dirs; i++) h_B[((size_t)s * n_dirs + i) * D + c] = (float)(acc[i] / n_quad);
        }
    }
    return MM_OK;
}
