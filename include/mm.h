/* include/mm.h — C ABI of the B200-native tensor-tomography gradient path (arxiv 2504.16446, "Mumott").
 *
 * Citations: P:NN = /root/reference/PAPER.md line NN.  Sx = reading x in DESIGN.md "Readings of the paper".
 *
 * What the library computes.  A sample is a grid of X*Y*Z voxels, each holding K basis coefficients
 * c[x][y][z][i] (Eq. 2).  For each of P goniometer settings s (rotation alpha_s, tilt beta_s,
 * R_s = R_beta R_alpha) and each raster position (j,k) of a J x Kd scan, the forward model is (Eq. 6)
 *
 *     I[s][j][k][c] = sum_xyz P_{sjk,xyz} sum_i B[s][i][c] c[x][y][z][i]
 *
 * where P_{sjk,xyz} is the John transform (Eq. 5) evaluated by Joseph's method with bilinear
 * interpolation of the field and B[s][i][c] is the segment-integrated basis matrix of Eq. 3.
 * The data term of Eq. 9 with residual r = Ac - I (Eq. 13) is L = 1/2 sum w r^2 (S10) and its
 * gradient is A^T (w r), A^T being the exact transpose of the discrete forward operator (S9).
 *
 * Conventions common to every call
 *   - All functions return mm_status and never throw.  mm_last_error() gives a thread-local message.
 *   - Arrays are dense, C order, fp32 unless stated.  Layouts:
 *       volume / gradient   [X][Y][Z][ldk]        channel stride ldk >= K floats ("c[x,y,z,i]")
 *       K-channel projection [P][J][Kd][ldk]
 *       sinogram, data, weights, wr  [P][J][Kd][D] (Table IV: data (n_j,n_k,n_phi) per projection)
 *       basis matrix B      [P][K][D]             (S3)
 *     Channels K..ldk-1 of INPUT arrays are ignored; of OUTPUT arrays they are written as 0.
 *   - "DEVICE" pointers are CUDA device memory on the current device, owned by the caller, not aliased with
 *     each other; the fast path needs ldk % 4 == 0 and 16-byte aligned bases, otherwise a slower scalar path
 *     runs (same results).  "HOST" pointers are ordinary host memory.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Device calls only enqueue
 *     work on it: no synchronisation, outputs overwritten (never accumulated).  The only memory a device call
 *     obtains itself is scratch from a memory pool the library owns (cudaMallocFromPoolAsync / cudaFreeAsync on
 *     `stream`: stream-ordered, no synchronisation, re-entrant, cached between calls; mm_workspace_release()
 *     returns it to the driver).
 *   - Volumes and data must be finite: taps outside the volume and rays with zero weight may still be read and
 *     multiplied by zero (a NaN there would spread).
 *   - mm_geometry is immutable after creation; calls on different streams may run concurrently.
 *   - Errors: NULL required pointer -> MM_ERR_NULL; K<1, ldk<K, D<1, D>MM_MAX_D, shape<1 -> MM_ERR_SHAPE;
 *     non-finite angle, non-orthonormal axes -> MM_ERR_VALUE; CUDA launch/alloc failures -> MM_ERR_CUDA /
 *     MM_ERR_ALLOC.  No CPU fallback exists anywhere in this library.
 */
#ifndef MM_H_
#define MM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MM_MAX_D 32          /* most detector segments the kernels hold in registers */

typedef enum {
    MM_OK = 0,
    MM_ERR_NULL = 1,
    MM_ERR_SHAPE = 2,
    MM_ERR_VALUE = 3,
    MM_ERR_ALLOC = 4,
    MM_ERR_CUDA = 5,
    MM_ERR_UNSUPPORTED = 6
} mm_status;

typedef struct mm_geometry mm_geometry;      /* opaque */

/* Acquisition geometry (Table I, Table IV, Eq. 4).  HOST memory, borrowed for
 * the duration of mm_geometry_create only.  A direction given as (0,0,0) takes its Table I standard value. */
typedef struct {
    int32_t volume_shape[3];     /* X, Y, Z  (Table IV volume_shape)                                        */
    int32_t det_shape[2];        /* J, Kd    (raster points along j and k)                                  */
    int32_t n_proj;              /* P                                                                       */
    const double *rotations;     /* [P] inner angle alpha_s, radians                                        */
    const double *tilts;         /* [P] outer angle beta_s, radians                                         */
    const double *j_offsets;     /* [P] delta j_s in raster steps (Eq. 4), NULL = 0                         */
    const double *k_offsets;     /* [P] delta k_s, NULL = 0                                                 */
    double p_dir[3];             /* beam direction p,           standard +z                                 */
    double j_dir[3];             /* raster direction j,         standard +y (S1)                            */
    double k_dir[3];             /* raster direction k,         standard +x (S1)                            */
    double q0_dir[3];            /* detector direction phi=0,   standard +x  (basis helper only)            */
    double q90_dir[3];           /* detector direction phi=90,  standard +y  (basis helper only)            */
    double inner_axis[3];        /* rotation axis alpha-hat,    standard +y                                 */
    double outer_axis[3];        /* tilt axis beta-hat,         standard +x                                 */
    double voxel_size;           /* a of Eq. 4, 0 = 1                                                       */
    double pixel_size;           /* b of Eq. 4, 0 = 1                                                       */
} mm_geometry_desc;

/* Build the per-projection ray table (host, fp64) and upload it to the current CUDA device.  For each s:
 * d_s = R_s^T p, j_s = R_s^T j, k_s = R_s^T k (sample frame); Joseph major axis m_s = lowest
 * index with |d_i| >= max|d| - 1e-6 (S8); step w_s = a/|d_m| (S7); the affine maps (j,k,n) -> in-slab position
 * and voxel -> detector position that follow from Eq. 4 with rotation centre (shape-1)/2 and detector centre
 * (det-1)/2 (S4).  The library owns *out; free with mm_geometry_destroy. */
mm_status mm_geometry_create(const mm_geometry_desc *desc, mm_geometry **out);
mm_status mm_geometry_destroy(mm_geometry *g);

/* Test introspection: sample-frame beam direction d, raster axes js, ks, major axis and Joseph step of
 * projection s (all HOST outputs; any may be NULL). */
mm_status mm_geometry_get(const mm_geometry *g, int32_t s, double d[3], double js[3], double ks[3],
                          int32_t *major_axis, double *step);

/* HOST helper, Eq. 3 for real spherical harmonics of even degree l <= ell_max,
 * 4pi-normalised, order l ascending then m = -l..l (S14), small-angle q(phi) = cos(phi) q0 + sin(phi) q90
 * (Eq. 1 second line): h_B[s][i][c] = mean over [seg_start[c], seg_end[c]] of
 * Y_i(R_s^T q(phi)), integrated exactly (the integrand is a trigonometric polynomial of degree <= ell_max, S15).
 * K = (ell_max+1)(ell_max+2)/2.  seg_start/seg_end: [D] radians, HOST.  h_B: [P][K][D] fp32, HOST, caller-owned. */
mm_status mm_basis_sh_matrix(const mm_geometry *g, int32_t ell_max, int32_t D, const double *seg_start,
                             const double *seg_end, float *h_B);

/* NEXT-4 — as mm_basis_sh_matrix with the full scattering vector of Eq. 1, first line (wide-angle scattering):
 * q(phi) = cos(2theta/2)(cos(phi) q0 + sin(phi) q90) - sin(2theta/2) p, two_theta in radians (0 = small-angle line).
 * Y_i(R_s^T q(phi)) is still a trigonometric polynomial of degree <= ell_max in phi: integrated exactly. */
mm_status mm_basis_sh_matrix_2theta(const mm_geometry *g, int32_t ell_max, double two_theta, int32_t D,
                                    const double *seg_start, const double *seg_end, float *h_B);

/* NEXT-2 — HOST helper, Eq. 3 for basis sets defined by a grid of orientations: dirs [n_dirs][3] HOST,
 * sample-frame vectors (normalised here); K = n_dirs.
 *   MM_BASIS_NN  nearest-neighbour indicators: B_i(q) = 1 if |q.g_i| is the largest (first on ties), else 0
 *   MM_BASIS_GK  Gaussian kernels: B_i(q) = exp(-theta_i^2 / (2 sigma^2)), theta_i = arccos|q.g_i|
 * (distances between lines, the SAXS RSM being even in q: DESIGN.md reading S20).  h_B[s][i][c] = mean of
 * B_i(R_s^T q(phi)) over n_quad midpoints of [seg_start[c], seg_end[c]].  h_B [P][n_dirs][D] fp32 HOST. */
#define MM_BASIS_NN 1
#define MM_BASIS_GK 2
mm_status mm_basis_grid_matrix(const mm_geometry *g, int32_t kind, int32_t n_dirs, const double *dirs, double sigma,
                               int32_t D, const double *seg_start, const double *seg_end, int32_t n_quad, float *h_B);

/* John transform, Eq. 5 / P:314, ray-stationary Joseph: for every ray (s,j,k) and channel i < K
 *   proj[s][j][k][i] = w_s * sum_{n=0}^{N_m-1} bilinear(vol[slab n])(pu_n, pv_n)_i, zero outside the volume.
 * vol [X][Y][Z][ldk] DEVICE in; proj [P][J][Kd][ldk] DEVICE out. */
mm_status mm_john_forward(const mm_geometry *g, const float *vol, int32_t K, int32_t ldk, float *proj,
                          void *stream);

/* Exact transpose of mm_john_forward (S9), voxel-stationary gather:
 *   vol_out[x][i] = sum_s w_s sum_{(j,k)} Lambda(pu(s,j,k;x_m) - x_u) Lambda(pv - x_v) proj[s][j][k][i].
 * proj [P][J][Kd][ldk] DEVICE in; vol_out [X][Y][Z][ldk] DEVICE out (overwritten). */
mm_status mm_john_adjoint(const mm_geometry *g, const float *proj, int32_t K, int32_t ldk, float *vol_out,
                          void *stream);

/* Reciprocal-space map of Eq. 6 (inner sum) and its transpose, per pixel:
 *   forward: sino[s][j][k][c] = sum_i B[s][i][c] proj[s][j][k][i]
 *   adjoint: proj[s][j][k][i] = sum_c B[s][i][c] sino[s][j][k][c]
 * B [P][K][D] DEVICE; proj [P][J][Kd][ldk] DEVICE; sino [P][J][Kd][D] DEVICE. */
mm_status mm_basis_forward(const mm_geometry *g, const float *B, const float *proj, int32_t K, int32_t ldk,
                           int32_t D, float *sino, void *stream);
mm_status mm_basis_adjoint(const mm_geometry *g, const float *B, const float *sino, int32_t K, int32_t ldk,
                           int32_t D, float *proj, void *stream);

/* Full forward model I = A c (Eq. 6-7) and its transpose, fused: the K-channel projections stay in
 * registers and never touch HBM (cf. the paper's fused kernel).
 *   mm_forward: vol -> sino [P][J][Kd][D];   mm_adjoint: sino -> vol_out [X][Y][Z][ldk] (overwritten). */
mm_status mm_forward(const mm_geometry *g, const float *B, const float *vol, int32_t K, int32_t ldk, int32_t D,
                     float *sino, void *stream);
mm_status mm_adjoint(const mm_geometry *g, const float *B, const float *sino, int32_t K, int32_t ldk, int32_t D,
                     float *vol_out, void *stream);

/* NEXT-1 — the adjoint as the paper words it (Joseph's method "using bilinear interpolation of the field
 * for the forward and the projection for the adjoint"): voxel-driven, NOT the transpose of mm_john_forward
 * (reading S9).  For every voxel x and projection s, with (j0,k0) the detector position of x (Eq. 4),
 *   vol_out[x][i] = sum_s w_s * bilinear(proj[s])(j0, k0)_i,   pixels outside the detector count as 0.
 * mm_john_backproject: proj [P][J][Kd][ldk] DEVICE in -> vol_out [X][Y][Z][ldk] DEVICE out (overwritten).
 * mm_backproject: the same applied to basis^T sino, fused (sino [P][J][Kd][D] DEVICE in); this is the pair
 * (forward, back-projection) the paper's SIRT/MITRA iterations use. */
mm_status mm_john_backproject(const mm_geometry *g, const float *proj, int32_t K, int32_t ldk, float *vol_out,
                              void *stream);
mm_status mm_backproject(const mm_geometry *g, const float *B, const float *sino, int32_t K, int32_t ldk, int32_t D,
                         float *vol_out, void *stream);

/* One fused gradient evaluation (Eq. 9 data term with a = 2, Eq. 13; S10, S11):
 *   phase 1 (all rays):   r = (A vol) - data;  wr = weights * r;  *loss = 1/2 sum weights r^2
 *   phase 2 (all voxels): grad = A^T wr
 * data, weights [P][J][Kd][D] DEVICE in (weights NULL = all ones); grad [X][Y][Z][ldk] DEVICE out;
 * loss: DEVICE double, overwritten; wr_workspace [P][J][Kd][D] DEVICE scratch, holds wr on return. */
mm_status mm_loss_gradient(const mm_geometry *g, const float *B, const float *vol, int32_t K, int32_t ldk,
                           int32_t D, const float *data, const float *weights, float *grad, double *loss,
                           float *wr_workspace, void *stream);

/* NEXT-4 — robust regression (HuberLoss; reading S23): as mm_loss_gradient with the Huber function of the
 * residual, rho(r) = 1/2 r^2 for |r| <= delta, delta (|r| - delta/2) beyond:  *loss = sum weights rho(r),
 * wr_workspace = weights * clip(r, -delta, delta), grad = A^T wr_workspace.  delta > 0. */
mm_status mm_loss_gradient_huber(const mm_geometry *g, const float *B, const float *vol, int32_t K, int32_t ldk, int32_t D,
                                 const float *data, const float *weights, float delta, float *grad, double *loss,
                                 float *wr_workspace, void *stream);

/* Phase 1 of mm_loss_gradient alone: wr = weights * (A vol - data), *loss = 1/2 sum weights r^2; lets a caller
 * pair the forward with the back-projector of its choice (mm_adjoint or mm_backproject), as SIRT/MITRA do.
 * Same arguments as mm_loss_gradient; wr [P][J][Kd][D] DEVICE out. */
mm_status mm_residual_loss(const mm_geometry *g, const float *B, const float *vol, int32_t K, int32_t ldk, int32_t D,
                           const float *data, const float *weights, float *wr, double *loss, void *stream);

/* SIRT / MITRA building blocks (SIRT as preconditioned weighted least squares; reading S19).
 * mm_reciprocal: x[i] <- 1/x[i] where x[i] > floor, else 0 — turns row sums |A| 1 (mm_forward of an all-ones
 *   volume with |B|) into the weights W and column sums |A|' 1 into the preconditioner C; n floats, DEVICE, in place.
 * mm_axpy_precond: c[i] <- c[i] - eta * pre[i] * grad[i] — the preconditioned update c <- c - C (.) A'(W r). */
mm_status mm_reciprocal(float *x, int64_t n, float floor, void *stream);
mm_status mm_axpy_precond(float *c, const float *grad, const float *pre, float eta, int64_t n, void *stream);

/* NEXT-4 — derived quantities of a reconstructed SH coefficient volume, per voxel:
 *   mean [N]               Eq. 10, the isotropic intensity <f> (= coefficient 0 with the 4pi normalisation, S14)
 *   moments [N][6]         Eq. 11, M_ij = <q_i q_j f>, stored xx, yy, zz, xy, xz, yz
 *   eigenvalues [N][3]     of M, descending;  eigenvectors [N][3][3] unit row vectors in the same order (sign
 *                          arbitrary; arbitrary within a degenerate eigenspace)
 *   fa [N]                 Eq. 12, fractional anisotropy (0 where M = 0)
 * vol [X][Y][Z][ldk] DEVICE in, real SH of even l in the order of mm_basis_sh_matrix (K = 1 or K >= 6); every
 * output is DEVICE, N = X*Y*Z, and may be NULL to skip it. */
mm_status mm_derived_quantities(const mm_geometry *g, const float *vol, int32_t K, int32_t ldk, float *mean, float *moments,
                                float *eigenvalues, float *eigenvectors, float *fa, void *stream);

/* NEXT-2 — sparse reciprocal-space map (the sparse pipelines "use a modified version of the John transform that
 * calculates the reciprocal-space and real-space projection operations simultaneously within one kernel, using a
 * sparse approximation to the reciprocal-space mapping ... such as only mapping one basis function to each segment").
 * Reading S26: the approximation keeps, for every projection s and segment c, the n_keep coefficients B[s][i][c] of
 * largest magnitude (lowest i first among equals) and zeroes the others.
 *   mm_basis_sparsify       HOST: h_B [P][K][D] -> h_B_out (same shape; may not alias h_B); n_keep >= K copies.
 *   mm_sparse_plan_create   HOST h_B (already sparse: an NN basis, or the output of mm_basis_sparsify): records for every
 *                           projection the channels i with a non-zero row B[s][i][:] and uploads the lists.  The plan
 *                           belongs to (g, K, D) and must be rebuilt when the zero pattern of B changes.
 *   mm_sparse_plan_info     max / mean number of active channels per projection; counts [P] HOST or NULL.
 *   mm_forward_sparse       = mm_forward with that B, marching only the active channels of each projection.
 *   mm_loss_gradient_sparse = mm_loss_gradient with that B: sparse phase 1, dense tensor-core contraction in phase 2.
 * B (DEVICE) must have the zero pattern the plan was made from: rows outside the lists are never read.  Results equal
 * the dense calls' on the same B to fp32 rounding.
 * With at most 32 active channels per projection the march runs on channel-planar, zero-padded copies of `vol` that the
 * call makes itself in the library's scratch pool (K planes of (X+4)(Y+4)(Z+4) floats, one set per family of major
 * axes in use: up to 2.2 x the volume), so that only the active channels' planes are read; otherwise, or if the pool
 * cannot supply the copies, it runs on `vol` as it is (same results to rounding, no scratch). */
typedef struct mm_sparse_plan mm_sparse_plan;
mm_status mm_basis_sparsify(const float *h_B, int32_t P, int32_t K, int32_t D, int32_t n_keep, float *h_B_out);
mm_status mm_sparse_plan_create(const mm_geometry *g, const float *h_B, int32_t K, int32_t D, mm_sparse_plan **out);
mm_status mm_sparse_plan_destroy(mm_sparse_plan *plan);
mm_status mm_sparse_plan_info(const mm_sparse_plan *plan, int32_t *max_active, double *mean_active, int32_t *counts);
mm_status mm_forward_sparse(const mm_geometry *g, const mm_sparse_plan *plan, const float *B, const float *vol, int32_t K,
                            int32_t ldk, int32_t D, float *sino, void *stream);
mm_status mm_loss_gradient_sparse(const mm_geometry *g, const mm_sparse_plan *plan, const float *B, const float *vol, int32_t K,
                                  int32_t ldk, int32_t D, const float *data, const float *weights, float *grad, double *loss,
                                  float *wr_workspace, void *stream);

/* NEXT-3 — regulariser and optimizer building blocks for a device-resident iteration.
 * mm_laplacian: vol_out[x][i] = sum of the six face neighbours of vol[x][i] - 6 vol[x][i], neighbours outside the
 *   volume counting as 0 (reading S21); vol, vol_out [X][Y][Z][ldk] DEVICE, distinct; pad channels written 0.
 *   The gradient of the Laplacian regulariser mu/2 ||Lap c||^2 is mu Lap(Lap c): two calls; of the L2Norm
 *   mu/2 ||c||^2 it is mu c: mm_axpy(grad, c, -mu, n).
 * mm_nesterov_step: v <- momentum v - eta grad;  c <- c + v  (GradientDescent with Nesterov momentum; the
 *   caller evaluates grad at c + momentum v, reading S22); n floats each, DEVICE. */
mm_status mm_laplacian(const mm_geometry *g, const float *vol, int32_t K, int32_t ldk, float *vol_out, void *stream);

/* The other regularisers of P:336-338 (reading S24; h(t) = t^2/(2 delta) for |t| <= delta, |t| - delta/2 beyond):
 *   MM_REG_L1     L1Norm         R = sum |c|,                  grad = sign(c)               (delta ignored)
 *   MM_REG_HUBER  HuberNorm      R = sum h(c),                 grad = clip(c/delta, -1, 1)
 *   MM_REG_TV     TotalVariation R = sum_x,i h(|D c_i(x)|),    grad = D^T (D c_i / max(|D c_i|, delta)),
 *                 D = forward differences along x, y, z (0 across the last face), per channel i.
 * vol [X][Y][Z][ldk] DEVICE in; grad_out same shape, DEVICE out (overwritten, pad channels 0), distinct from vol;
 * value: DEVICE double, overwritten with R, or NULL. */
#define MM_REG_L1 1
#define MM_REG_HUBER 2
#define MM_REG_TV 3
mm_status mm_regulariser(const mm_geometry *g, int32_t kind, const float *vol, int32_t K, int32_t ldk, float delta,
                         float *grad_out, double *value, void *stream);
mm_status mm_nesterov_step(float *c, float *v, const float *grad, float eta, float momentum, int64_t n, void *stream);

/* NEXT-3 — the whole regularised iteration on the device (MITRA = gradient descent with Nesterov momentum and
 * regularisers, SIGTT "uses a stop criterion based on the relative change of the loss function"; the
 * asynchronous pipelines keep the loop on the GPU).  Reading S25: iteration k = 0, 1, ... works at the look-ahead point
 * y_k = c_k + m v_k,
 *     L_k = 1/2 sum w (A y_k - data)^2 + mu_laplacian/2 ||Lap y_k||^2 + mu_l2/2 ||y_k||^2,   g_k = its gradient at y_k,
 *     v_{k+1} = m v_k - eta g_k,    c_{k+1} = c_k + v_{k+1},
 * and after the update of every check_every-th iteration (k + 1 a multiple of check_every, k >= 1) stops if
 * |L_k - L_{k-1}| <= tol |L_k| (tol <= 0: never).  c, v [X][Y][Z][ldk] DEVICE, in/out (v = momentum state: zeros for a
 * fresh start; channels K..ldk-1 are left alone); losses DEVICE double[max_iter], out (L_0 .. L_{n_iter-1}); n_iter HOST
 * out = iterations done.  All work is enqueued on `stream`; per check the host reads one 4-byte flag and waits for
 * the stream (the only synchronisation; with tol <= 0 the call is fully asynchronous).  Scratch (2 or 4 volumes and
 * one sinogram) comes from the library's stream-ordered pool.  MM_ERR_VALUE for eta <= 0, negative momentum/weights,
 * max_iter or check_every < 1. */
typedef struct {
    float eta;              /* step length                                                      */
    float momentum;         /* Nesterov m, 0 = plain gradient descent                   */
    float mu_laplacian;     /* weight of the Laplacian regulariser, 0 = off            */
    float mu_l2;            /* weight of the L2Norm regulariser, 0 = off               */
    int32_t max_iter;
    int32_t check_every;
    double tol;
} mm_iterate_params;
mm_status mm_iterate(const mm_geometry *g, const float *B, int32_t K, int32_t ldk, int32_t D, const float *data,
                     const float *weights, const mm_iterate_params *params, float *c, float *v, double *losses,
                     int32_t *n_iter, void *stream);

/* Fixed-step gradient-descent update c <- c - eta * grad on n floats (GradientDescent); DEVICE. */
mm_status mm_axpy(float *c, const float *grad, float eta, int64_t n, void *stream);

/* End-to-end convenience with HOST buffers (what a caller without device memory uses): copies B, vol, data,
 * weights host->device, runs mm_loss_gradient, copies grad and loss back, and synchronises.  All pointers
 * HOST (pinned memory makes the copies asynchronous DMA); h_weights may be NULL; h_loss is one double.
 * The device workspace (one arena of 2 volumes + 2-3 sinograms + B, and one stream) is owned by the library,
 * grows on demand, is reused by later calls and is freed by mm_host_workspace_release(); calls are serialised
 * inside the library.  MM_ERR_ALLOC if the arena cannot be allocated (nothing is left allocated then). */
mm_status mm_host_workspace_release(void);
/* Also returns to the driver the device memory cached in the library's stream-ordered scratch pool (see "stream"
 * above): the adjoint's split operand tiles (P*ldk*D*8 bytes), the forward's repacked volume when ldk = 48 (one
 * volume), the sparse forward's channel-planar copies, mm_iterate's work arrays.  The pool refills on the next call
 * that needs it. */
mm_status mm_workspace_release(void);
mm_status mm_loss_gradient_host(const mm_geometry *g, const float *h_B, const float *h_vol, int32_t K,
                                int32_t ldk, int32_t D, const float *h_data, const float *h_weights,
                                float *h_grad, double *h_loss);

/* A^T (a6 + a7) for callers that may not allocate: code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc.  Same arguments, kernels (bop_prep_kernel + adjoint_brick_kernel) and result as
 * mm_adjoint on the shapes the brick kernel serves, but the one piece of scratch it needs — the split operand tiles
 * of w_s B_s, P * 2 * npad(ldk) * D * 4 bytes with npad = ldk rounded up to 16/32/48/64/96/128/192 — lives in a
 * static device array of MM_ADJOINT_NOALLOC_MAX_BYTES inside the library (held on every GPU that loads it until the
 * process exits) instead of the stream-ordered pool.  The call makes no cudaMalloc/cudaFree/pool call of any kind.
 *   - MM_ERR_UNSUPPORTED (nothing enqueued) if the scratch would exceed the maximum, or the shape is not the brick
 *     kernel's: D = 8 or 16, ldk % 4 == 0, ldk <= 192, 16-byte aligned B / sino / vol_out, a geometry whose brick
 *     shadow fits a 16 x 17 pixel tile (every standard tomographic geometry).  There is no fallback: use mm_adjoint.
 *     Config 5 needs 1.1 MB (P = 360, ldk = 48, D = 8), config 4 2.0 MB (P = 500, ldk = 32, D = 16).
 *   - All calls share the array.  Every element the kernel reads is rewritten by the call itself, so a call never
 *     sees an earlier call's contents; but two calls whose kernels can overlap on the GPU (different streams, no
 *     dependency) race on it: serialise them (one stream, or an event between them).
 *   - vol_out [X][Y][Z][ldk] is overwritten; asynchronous on `stream` like every device call here. */
#define MM_ADJOINT_NOALLOC_MAX_BYTES (4u << 20)
mm_status mm_adjoint_noalloc(const mm_geometry *g, const float *B, const float *sino, int32_t K, int32_t ldk,
                             int32_t D, float *vol_out, void *stream);

/* Number of kernel launches this library has enqueued since load (for bench accounting). */
int64_t mm_launch_count(void);

/* Measurement hook: if `cuda_event` (a cudaEvent_t passed as void*) is non-NULL, later mm_loss_gradient calls
 * made by this host thread record it on their stream between phase 1 and phase 2, so a caller can time the
 * two kernels of one call separately.  NULL clears the hook.  Does not change what is computed. */
mm_status mm_set_phase_event(void *cuda_event);

const char *mm_status_string(mm_status s);
const char *mm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MM_H_ */
