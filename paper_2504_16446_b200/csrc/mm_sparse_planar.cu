// mm_sparse_planar.cu — NEXT-2, second cut: the sparse forward on CHANNEL-PLANAR copies of the volume.
//
// mm_sparse.cu marches the caller's [voxel][ldk] volume with a lane per active channel: 18 scattered 4-byte reads of a
// 672-byte record (K = 162) still touch 18 of its 21 sectors, so sparsity saved register traffic but not HBM or L2
// bytes (24.9 ms against 39.9 ms dense on the 100^3 / 240-projection / 162-direction case).  Here the
// volume is first transposed into one padded 3-D plane per channel, and a THREAD owns a ray: the 32 lanes of a warp
// are 32 neighbouring rays along k, which for every tap read 32 neighbouring floats of ONE plane — a 128-byte
// wavefront — and only the planes of the projection's active channels are read at all (18.5 of 162 on average: an
// 80 MB working set per projection, which stays in L2).
//   copy Z: planes [K][X+4][Y+4][Z+4], z fastest   (major axis x or y: neighbouring rays along k differ mainly in z)
//   copy X: planes [K][Z][Y+4][X+4],   x fastest   (major axis z: they differ mainly in x)
// Two zero voxels pad every in-slab axis, so no tap needs a bounds test and the four taps of a slab sit at fixed
// offsets (0, 1, row, row + 1) from one base.  Arithmetic as in the dense ldk = 48 march: 24.40 fixed-point positions,
// nested-difference bilinear form, fp32 rounds of 4 slabs flushed into fp64 totals, fp64 epilogue (Eq. 6, 13, 9).
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <string>

#include "mm_internal.h"

#ifndef PL_MINB_HI
#define PL_MINB_HI 3                    // resident 128-thread blocks per SM asked of the compiler beyond 16 active channels
#endif
#ifndef PL_CB
#define PL_CB 2                         // channels whose 16 taps (4 slabs) are in flight together; divides 8
#endif

namespace {

constexpr int PAD = 2;                  // zero voxels on each side of an in-slab axis (the range clip leaves half a slab, |slope| <= 1)
#define PL_FX_BITS 40
#define PL_FX_ONE 1099511627776.0
#define PL_FX_INV 2.3283064365386963e-10f

// Transpose 32 voxels that are consecutive along the copy's fastest axis: read their records (ldk floats each,
// coalesced) into shared memory, write one 128-byte segment per channel.  XFAST = 0: copy Z (segment along z);
// XFAST = 1: copy X (segment along x).  The planes were zeroed before (padding).
template <int XFAST>
__global__ void __launch_bounds__(256) planar_copy_kernel(const float *__restrict__ src, float *__restrict__ dst, int X, int Y, int Z, int K, int ldk)
{
    extern __shared__ float tile[];                               // [32][ldk + 1]
    const int pitch = ldk + 1;
    const int nseg = XFAST ? (X + 31) / 32 : (Z + 31) / 32;       // segments per line of the fastest axis
    const long long line = blockIdx.x / nseg;                     // copy Z: (x, y); copy X: (z, y)
    const int f0 = (int)(blockIdx.x % nseg) * 32;
    const int a = (int)(line / Y), y = (int)(line % Y);           // copy Z: a = x; copy X: a = z
    const int nf = min(32, (XFAST ? X : Z) - f0);
    for (int i = threadIdx.x; i < nf * ldk; i += 256) {
        const int v = i / ldk, c = i - v * ldk;
        const long long vox = XFAST ? ((long long)(f0 + v) * Y + y) * Z + a : ((long long)a * Y + y) * Z + f0 + v;
        tile[v * pitch + c] = __ldg(src + vox * ldk + c);
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const long long plane = XFAST ? (long long)Z * (Y + 2 * PAD) * (X + 2 * PAD) : (long long)(X + 2 * PAD) * (Y + 2 * PAD) * (Z + 2 * PAD);
    const long long row = XFAST ? ((long long)a * (Y + 2 * PAD) + y + PAD) * (X + 2 * PAD) + f0 + PAD
                                : ((long long)(a + PAD) * (Y + 2 * PAD) + y + PAD) * (Z + 2 * PAD) + f0 + PAD;
    if (lane < nf)
        for (int k = w; k < K; k += 8) dst[k * plane + row + lane] = tile[lane * pitch + k];
}

struct PlanarArgs {
    const MMProj *tab;
    const float *volZ, *volX;       // the planar copies (NULL where no projection needs one)
    const int *idx, *count;         // the plan's active-channel lists
    int slots;
    int K, X, Y, Z, J, Kd, P, D;
    const float *B, *data, *weights;
    float *sino;                    // MODE 1: model sinogram; MODE 2: wr
    double *loss;
};

__device__ __forceinline__ void pl_clip(double A, double s, int N, double &lo, double &hi)
{
    if (fabs(s) < 1e-12) {
        if (!(A > -1.0 && A < (double)N)) hi = lo - 1.0;
        return;
    }
    double t0 = (-1.0 - A) / s, t1 = ((double)N - A) / s;
    if (t0 > t1) { const double t = t0; t0 = t1; t1 = t; }
    lo = fmax(lo, t0 - 0.5);        // half a slab to spare: positions stay within (-1.5, N + 0.5), inside the padding
    hi = fmin(hi, t1 + 0.5);
}

__device__ __forceinline__ float ldg_nc_f32(const float *p)
{
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}

// A thread owns a ray (lane = k within a tile of 32, warp = j within a tile of 4); NA = active channels, rounded up.
template <int NA, int DMAX, int MODE>
__global__ void __launch_bounds__(128, NA <= 16 ? 4 : PL_MINB_HI) john_forward_planar_kernel(const PlanarArgs a)
{
    constexpr int TK = 32, TJ = 4;
    const int tid = threadIdx.x, lane = tid & 31, wj = tid >> 5;
    const int tiles_k = (a.Kd + TK - 1) / TK, tiles_j = (a.J + TJ - 1) / TJ;
    const int tpp = tiles_k * tiles_j;
    const int s = blockIdx.x / tpp;
    const int tile = blockIdx.x - s * tpp;
    const int tk = tile % tiles_k, tj = tile / tiles_k;
    const int j = tj * TJ + wj, k = tk * TK + lane;
    const bool ray_ok = (j < a.J) && (k < a.Kd);
    const MMProj *pg = a.tab + s;
    const int m = pg->m;
    const int Nm = (m == 0) ? a.X : (m == 1 ? a.Y : a.Z);
    const int Nu = (m == 0) ? a.Y : a.X, Nv = (m == 2) ? a.Y : a.Z;
    const int DX = a.X + 2 * PAD, DY = a.Y + 2 * PAD, DZ = a.Z + 2 * PAD;
    // strides (floats) inside a plane; the unit-stride in-slab axis is v (copy Z) or u (copy X)
    const int sM = (m == 0) ? DY * DZ : (m == 1 ? DZ : DY * DX);
    const int sU = (m == 0) ? DZ : (m == 1 ? DY * DZ : 1);
    const int sV = (m == 2) ? DX : 1;
    const int sR = (m == 2) ? sV : sU;                            // the in-slab axis that is not unit-stride
    const int o0 = (m == 2) ? PAD * DX + PAD : (PAD * DY + PAD) * DZ + PAD;
    const long long plane = (m == 2) ? (long long)a.Z * DY * DX : (long long)DX * DY * DZ;
    const float *const vol = (m == 2) ? a.volX : a.volZ;
    const int na = a.count[s];

    __shared__ long long s_plane[NA];                             // element offset of each active channel's plane
    __shared__ int s_ch[NA];                                      // and the channel itself
    __shared__ int s_range[2];
    if (tid < NA) {
        s_ch[tid] = (tid < na) ? a.idx[(long long)s * a.slots + tid] : 0;
        s_plane[tid] = (long long)s_ch[tid] * plane;
    }
    if (tid == 0) { s_range[0] = 0x7fffffff; s_range[1] = -1; }

    int n0 = 0, n1 = -1;
    double Au = 0.0, Av = 0.0;
    if (ray_ok) {
        Au = pg->Cu + (double)j * pg->Mju + (double)k * pg->Mku;
        Av = pg->Cv + (double)j * pg->Mjv + (double)k * pg->Mkv;
        double lo = 0.0, hi = (double)(Nm - 1);
        pl_clip(Au, pg->su, Nu, lo, hi);
        pl_clip(Av, pg->sv, Nv, lo, hi);
        n0 = (int)ceil(lo); n1 = (int)floor(hi);
    }
    __syncthreads();
    if (n1 >= n0) { atomicMin(&s_range[0], n0); atomicMax(&s_range[1], n1); }
    __syncthreads();
    // all rays of the block march the union of their slab ranges in step (a slab outside a ray's own range reads
    // element 0 of the plane, which is padding, as are its three neighbours)
    const int nbeg = s_range[0], nend = s_range[1];
    const int rounds = (nend >= nbeg) ? (nend - nbeg + 4) / 4 : 0;
    const long long su_fx = pg->su_fx, sv_fx = pg->sv_fx;
    long long pu = (long long)floor(Au * PL_FX_ONE) + (long long)nbeg * su_fx;
    long long pv = (long long)floor(Av * PL_FX_ONE) + (long long)nbeg * sv_fx;
    int on = o0 + nbeg * sM;
    int n = nbeg;

    float acc[NA];
    double tot[NA];
#pragma unroll
    for (int i = 0; i < NA; i++) { acc[i] = 0.f; tot[i] = 0.0; }

    for (int rd = 0; rd < rounds; rd++) {
        int o[4];
        float f1[4], f2[4];                                       // fractions along the unit-stride axis and along the other one
#pragma unroll
        for (int i = 0; i < 4; i++) {
            const int iu = (int)(pu >> PL_FX_BITS), iv = (int)(pv >> PL_FX_BITS);
            const float fu = (float)(unsigned int)(pu >> (PL_FX_BITS - 32)) * PL_FX_INV;
            const float fv = (float)(unsigned int)(pv >> (PL_FX_BITS - 32)) * PL_FX_INV;
            o[i] = (n + i >= n0 && n + i <= n1) ? on + iu * sU + iv * sV : 0;
            f1[i] = (m == 2) ? fu : fv;
            f2[i] = (m == 2) ? fv : fu;
            pu += su_fx; pv += sv_fx; on += sM;
        }
        n += 4;
#pragma unroll
        for (int g = 0; g < NA; g += PL_CB) {
            if (g < na) {                                         // uniform over the block
                float c[PL_CB][4][4];
#pragma unroll
                for (int e = 0; e < PL_CB; e++) {
                    const float *pl = vol + s_plane[g + e];       // (a slot past na reads plane 0 and is never used)
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        const float *p = pl + o[i];
                        c[e][i][0] = ldg_nc_f32(p);
                        c[e][i][1] = ldg_nc_f32(p + 1);
                        c[e][i][2] = ldg_nc_f32(p + sR);
                        c[e][i][3] = ldg_nc_f32(p + sR + 1);
                    }
                }
#pragma unroll
                for (int e = 0; e < PL_CB; e++)
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        const float a0 = fmaf(f1[i], c[e][i][1] - c[e][i][0], c[e][i][0]);
                        const float a1 = fmaf(f1[i], c[e][i][3] - c[e][i][2], c[e][i][2]);
                        acc[g + e] += fmaf(f2[i], a1 - a0, a0);
                    }
            }
        }
#pragma unroll
        for (int i = 0; i < NA; i++) { tot[i] += (double)acc[i]; acc[i] = 0.f; }
    }

    // reciprocal-space map restricted to the active rows of B_s (Eq. 6), residual, loss: fp64, all in this thread
    const double w = pg->w64;
    double part[DMAX];
#pragma unroll
    for (int c = 0; c < DMAX; c++) part[c] = 0.0;
    const float *Bs = a.B + (long long)s * a.K * a.D;
#pragma unroll
    for (int i = 0; i < NA; i++) {
        if (i < na) {
            const int ch = s_ch[i];
            const double pv_ = w * tot[i];
#pragma unroll
            for (int c = 0; c < DMAX; c++)
                if (c < a.D) part[c] = fma((double)__ldg(Bs + (long long)ch * a.D + c), pv_, part[c]);
        }
    }
    double lsum = 0.0;
    if (ray_ok) {
        const long long ray = ((long long)s * a.J + j) * a.Kd + k;
#pragma unroll
        for (int c = 0; c < DMAX; c++) {
            if (c < a.D) {
                const long long oo = ray * a.D + c;
                if (MODE == 1) {
                    a.sino[oo] = (float)part[c];
                } else {
                    const double res = part[c] - (double)__ldg(a.data + oo);
                    const double wt = a.weights ? (double)__ldg(a.weights + oo) : 1.0;
                    a.sino[oo] = (float)(wt * res);
                    lsum += 0.5 * wt * res * res;
                }
            }
        }
    }
    if (MODE == 2) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) lsum += __shfl_xor_sync(0xffffffffu, lsum, off);
        __shared__ double red[4];
        if (lane == 0) red[wj] = lsum;
        __syncthreads();
        if (tid == 0) {
            const double t = red[0] + red[1] + red[2] + red[3];
            if (t != 0.0) atomicAdd(a.loss, t);
        }
    }
}

template <int MODE>
cudaError_t launch_planar(const PlanarArgs &a, int max_active, cudaStream_t st)
{
    const long long tiles = (long long)a.P * ((a.J + 3) / 4) * ((a.Kd + 31) / 32);
#define MM_PL_CASE(NA, DM) john_forward_planar_kernel<NA, DM, MODE><<<(unsigned)tiles, 128, 0, st>>>(a)
#define MM_PL_D(DM) do { if (max_active <= 8) MM_PL_CASE(8, DM); else if (max_active <= 16) MM_PL_CASE(16, DM); \
                         else if (max_active <= 24) MM_PL_CASE(24, DM); else MM_PL_CASE(32, DM); } while (0)
    if (a.D <= 8) MM_PL_D(8); else if (a.D <= 16) MM_PL_D(16); else MM_PL_D(32);
#undef MM_PL_D
#undef MM_PL_CASE
    return cudaGetLastError();
}

}  // namespace

bool mm_sparse_planar_supported(const mm_geometry *g, int K, int ldk, int max_active)
{
    const long long DX = g->shape[0] + 2 * PAD, DY = g->shape[1] + 2 * PAD, DZ = g->shape[2] + 2 * PAD;
    return max_active >= 1 && max_active <= 32 && K <= ldk && ldk <= 256 && DX * DY * DZ < (1LL << 31) &&
           (size_t)32 * (ldk + 1) * sizeof(float) <= 48 * 1024;
}

// Transposes `vol` into the planar copies the geometry needs (pooled scratch, stream-ordered) and runs the march.
// mode 1: sino = model sinogram; mode 2: sino = wr, *loss += L.  Returns a cudaError_t; on failure nothing useful was
// enqueued and the caller takes the record-layout kernel of mm_sparse.cu.
int mm_sparse_planar_launch(const mm_geometry *g, const int *d_idx, const int *d_count, int slots, int max_active, const float *B,
                            const float *vol, int K, int ldk, int D, const float *data, const float *weights, float *sino,
                            double *loss, int mode, void *stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    const int X = g->shape[0], Y = g->shape[1], Z = g->shape[2];
    int axis[3] = {0, 0, 0};
    for (const MMProj &t : g->table) axis[t.m]++;
    const bool needZ = axis[0] + axis[1] > 0, needX = axis[2] > 0;
    const size_t planeZ = (size_t)(X + 2 * PAD) * (Y + 2 * PAD) * (Z + 2 * PAD), planeX = (size_t)Z * (Y + 2 * PAD) * (X + 2 * PAD);
    float *cZ = nullptr, *cX = nullptr;
    cudaError_t e = cudaSuccess;
    if (needZ) e = mm_scratch_alloc((void **)&cZ, planeZ * K * sizeof(float), st);
    if (e == cudaSuccess && needX) e = mm_scratch_alloc((void **)&cX, planeX * K * sizeof(float), st);
    int copies = 0;
    const size_t smem = (size_t)32 * (ldk + 1) * sizeof(float);
    if (e == cudaSuccess && needZ) {
        e = cudaMemsetAsync(cZ, 0, planeZ * K * sizeof(float), st);
        if (e == cudaSuccess) {
            planar_copy_kernel<0><<<(unsigned)((long long)X * Y * ((Z + 31) / 32)), 256, smem, st>>>(vol, cZ, X, Y, Z, K, ldk);
            e = cudaGetLastError(); copies++;
        }
    }
    if (e == cudaSuccess && needX) {
        e = cudaMemsetAsync(cX, 0, planeX * K * sizeof(float), st);
        if (e == cudaSuccess) {
            planar_copy_kernel<1><<<(unsigned)((long long)Z * Y * ((X + 31) / 32)), 256, smem, st>>>(vol, cX, X, Y, Z, K, ldk);
            e = cudaGetLastError(); copies++;
        }
    }
    if (e == cudaSuccess) {
        PlanarArgs a;
        a.tab = g->d_table; a.volZ = cZ; a.volX = cX; a.idx = d_idx; a.count = d_count; a.slots = slots;
        a.K = K; a.X = X; a.Y = Y; a.Z = Z; a.J = g->J; a.Kd = g->Kd; a.P = g->P; a.D = D;
        a.B = B; a.data = data; a.weights = weights; a.sino = sino; a.loss = loss;
        e = (mode == 1) ? launch_planar<1>(a, max_active, st) : launch_planar<2>(a, max_active, st);
        if (e == cudaSuccess) mm_note_launches(copies + 1);
    }
    if (cZ) mm_scratch_free(cZ, st);
    if (cX) mm_scratch_free(cX, st);
    return (int)e;
}
