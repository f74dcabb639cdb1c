// mm_internal.h — private to the CUDA library (never included by oracle/).
#pragma once
#include <stddef.h>
#include <stdint.h>

#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "mm.h"

// Per-projection ray table entry, built on the host in fp64 (mm_geometry.cpp), read by every kernel.
//
// Forward (ray-stationary Joseph; Eq. 4): ray (j,k) of projection s crosses
// slab n of the major axis m at in-slab position
//     pu = Cu + j*Mju + k*Mku + n*su,      pv = Cv + j*Mjv + k*Mkv + n*sv         (voxel units)
// The kernels evaluate this in 24.40 fixed point (exact incremental adds along the ray), hence the *_fx
// copies of the slopes.
//
// Adjoint (voxel-stationary gather): voxel (x,y,z) projects to detector position
//     j0 = Jc + Jx.x,   k0 = Kc + Kx.x
// and a ray displaced by (dj,dk) from there passes the voxel's slab at in-slab displacement
//     du = Mju*dj + Mku*dk,   dv = Mjv*dj + Mkv*dk;   weight = w * Lambda(du) * Lambda(dv).
// Non-zero weights need |dj| < hj, |dk| < hk (bounding box of M^-1 (-1,1)^2).
struct MMProj {
    double Cu, Mju, Mku, su;
    double Cv, Mjv, Mkv, sv;
    // --- 96 contiguous bytes read as one block by the tensor-core adjoint (struct TcProj in mm_adjoint_tc.cu) ---
    double Jc, Jx[3];
    double Kc, Kx[3];
    float mju, mku, mjv, mkv;      // fp32 copies for the adjoint weights
    float hj, hk;                  // candidate window half-widths
    float w;                       // Joseph step a/|d_m|
    int gcode;                     // gather window: 1 = generic loop; 4 + 2*(NJ-2) + (NK-2) = fixed NJ x NK, NJ,NK in {2,3}
    // ---
    long long su_fx, sv_fx;        // round(su * 2^40), round(sv * 2^40)
    double w64;                    // Joseph step a/|d_m| unrounded (forward epilogue)
    int m, u, v;                   // major axis and the two in-slab axes (u < v)
    int pad_;
};
static_assert(offsetof(MMProj, gcode) - offsetof(MMProj, Jc) == 92, "gather block of MMProj must be 96 contiguous bytes");

struct MMProjHost {
    double R[9];                   // R_s, sample -> lab
    double d[3], js[3], ks[3];     // sample-frame beam direction and raster axes
    int m;
    double w;
};

struct mm_geometry {
    int32_t shape[3];
    int32_t J, Kd, P;
    double a, b;
    double q0[3], q90[3], p[3];
    std::vector<MMProjHost> host;
    std::vector<MMProj> table;
    MMProj *d_table;               // device copy of `table`
    int device;
    // detector tile (pixels) that holds every candidate ray of a 4x4x8 voxel brick, maximum over the projections;
    // 0 if some projection needs the generic candidate window or a tile beyond 16 x 17 (mm_adjoint_brick.cu)
    int brick_tj, brick_tk;
};

void mm_set_error(const std::string &msg);
void mm_note_launches(int n);          // kernels enqueued outside mm_kernels.cu (mm_launch_count accounting)

// Arguments of the voxel-stationary (adjoint) kernels.
struct AdjArgs {
    const MMProj *tab;
    const float *src;         // K-channel: proj [P][J][Kd][ldk]; fused: sino [P][J][Kd][D]
    const float *B;           // fused only
    float *out;               // [X][Y][Z][ldk]
    int K, ldk, D;
    int X, Y, Z, J, Kd, P;
    int vec_ok;               // fused: D % 4 == 0 and src 16-byte aligned
    long long vox_begin, vox_end;   // fused kernels: voxels [vox_begin, vox_end) of the launch (whole volume by default)
    int bilinear;             // 0: exact transpose of the Joseph forward (S9); 1: the paper's bilinear back-projection
};

// mm_runtime.cu: stream-ordered scratch from the library's own memory pool; TMA tensor maps
cudaError_t mm_scratch_alloc(void **p, size_t bytes, cudaStream_t st);
cudaError_t mm_scratch_free(void *p, cudaStream_t st);
void mm_scratch_trim();
bool mm_tma_available();
bool mm_tma_encode_4d_f32(void *tmap_out, const void *base, const unsigned long long n[4], const unsigned box[4], int swizzle);

// mm_adjoint_brick.cu: fused adjoint, voxel bricks + TMA-staged detector tiles + tcgen05 (3xTF32), the primary path
bool mm_adjoint_brick_supported(const mm_geometry *g, const AdjArgs &a);
int mm_adjoint_brick_launch(const mm_geometry *g, const AdjArgs &a, void *stream);   // returns a cudaError_t
// mm_sparse_planar.cu: the sparse forward on channel-planar copies of the volume (returns a cudaError_t)
bool mm_sparse_planar_supported(const mm_geometry *g, int K, int ldk, int max_active);
int mm_sparse_planar_launch(const mm_geometry *g, const int *d_idx, const int *d_count, int slots, int max_active, const float *B,
                            const float *vol, int K, int ldk, int D, const float *data, const float *weights, float *sino,
                            double *loss, int mode, void *stream);

// mm_adjoint_tc.cu: fused adjoint with the basis contraction on the tensor cores (tcgen05, 3xTF32).
bool mm_adjoint_tc_supported(const AdjArgs &a);
int mm_adjoint_tc_launch(const AdjArgs &a, void *stream);   // returns a cudaError_t
