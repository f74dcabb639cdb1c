// mm_kernels.cu — CUDA kernels (sm_100a) and C-ABI entry points of the tensor-tomography gradient path.
// Citations: P:NN = PAPER.md line NN; Sx = DESIGN.md reading x.  See include/mm.h for the contract.
//
// Kernel inventory
//   john_forward_kernel<VEC,G,NQ,DMAX,MODE>  ray-stationary Joseph march, lanes over channels;
//        MODE 0: write K-channel projections; MODE 1: fused basis map -> sinogram (Eq. 6);
//        MODE 2: fused basis map + residual + weighted loss (Eq. 13, Eq. 9) -> wr, loss
//   john_adjoint_kernel<VEC,G,NQ>            exact-transpose voxel gather of K-channel projections (S9)
//   adjoint_fused_kernel<KMAX,DMAX>          voxel gather of the D-channel sinogram, then B^T (Eq. 6 transposed)
//   basis_forward_kernel / basis_adjoint_kernel, axpy_kernel
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#include <atomic>
#include <mutex>
#include <string>

#include "mm_internal.h"

static std::atomic<long long> g_launches{0};

extern "C" int64_t mm_launch_count(void) { return (int64_t)g_launches.load(); }
void mm_note_launches(int n) { g_launches.fetch_add(n); }

static thread_local cudaEvent_t g_phase_event = nullptr;

extern "C" mm_status mm_set_phase_event(void *cuda_event)
{
    g_phase_event = (cudaEvent_t)cuda_event;
    return MM_OK;
}

#ifndef FWD_GS
#define FWD_GS 8                          // projections interleaved in block order (L2 reuse across projections)
#endif
#ifndef FWD_MINB
#define FWD_MINB 4
#endif
#ifndef FWD_U
#define FWD_U 2                         // slabs in flight per lane in the cooperative forward march
#endif
#ifndef FWD_U8
#define FWD_U8 8                        // same, for 32-byte lanes: a whole round of 8 slabs
#endif
#ifndef FWD_MINB8
#define FWD_MINB8 2                     // resident blocks per SM asked of the compiler for 32-byte lanes
#endif
#ifndef FWD_MIX48
#define FWD_MIX48 1
#endif
#ifndef FWD_COMMON_START
#define FWD_COMMON_START 1              // cooperative march: the rays of a block start at the block's first slab
#endif
#ifndef FWD_TK
#define FWD_TK 4                        // rays along k in the tile of a 32-ray block
#endif
// In-slab ray positions in 24.40 fixed point: exact incremental adds along the ray, slope resolution 2^-41 voxel per
// slab (2e-10 voxel over 256 slabs; 32.32 left 3e-8, a shear common to all rays of a projection and therefore a
// coherent error in the residual).  Integer part = tap index, top 32 fraction bits -> bilinear weight.
#define FX_BITS 40
#define FX_ONE 1099511627776.0         // 2^40
#define FX_INV 2.3283064365386963e-10f // 2^-32 (the weight is taken from the top 32 fraction bits)

// ================================================================================================
// forward: ray-stationary Joseph
// ================================================================================================
struct FwdArgs {
    const MMProj *tab;
    const float *vol;
    int zero_vox;             // LERP only: vol is the library's copy [N+1][ldk] whose last record (index N) is all zeros
    int K, ldk;
    int X, Y, Z, J, Kd, P;
    float *proj;              // MODE 0 out [P][J][Kd][ldk]
    const float *B;           // MODE 1,2 [P][K][D]
    int D;
    const float *data;        // MODE 2
    const float *weights;     // MODE 2 (may be NULL)
    float *sino;              // MODE 1: model sinogram; MODE 2: wr
    double *loss;             // MODE 2
    float huber;              // MODE 2: Huber threshold delta; <= 0 = squared loss
};

template <int VEC>
struct Ld;
template <>
struct Ld<4> {
    static __device__ __forceinline__ void ld(const float *p, float (&v)[4])
    {
        const float4 t = __ldg(reinterpret_cast<const float4 *>(p));
        v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
    }
    static __device__ __forceinline__ void st(float *p, const float (&v)[4])
    {
        *reinterpret_cast<float4 *>(p) = make_float4(v[0], v[1], v[2], v[3]);
    }
};
template <>
struct Ld<8> {                 // 256-bit accesses (sm_100: LDG.E.256 / STG.E.256); p must be 32-byte aligned
    static __device__ __forceinline__ void ld(const float *p, float (&v)[8])
    {
        asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
            : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]) : "l"(p));
    }
    static __device__ __forceinline__ void st(float *p, const float (&v)[8])
    {
        asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                     ::"l"(p), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]) : "memory");
    }
};
template <>
struct Ld<1> {
    static __device__ __forceinline__ void ld(const float *p, float (&v)[1]) { v[0] = __ldg(p); }
    static __device__ __forceinline__ void st(float *p, const float (&v)[1]) { *p = v[0]; }
};

// read-only 16-byte load that the compiler may not sink below later loads (keeps FWD_U slabs in flight)
__device__ __forceinline__ float4 ldg_nc_v4(const float4 *p)
{
    float4 v;
    asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// VEC floats (16 or 32 bytes) through the read-only path, in program order like ldg_nc_v4
template <int VEC>
__device__ __forceinline__ void ldg_nc_vec(const float *p, float (&v)[VEC])
{
    if constexpr (VEC == 4) {
        asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]) : "l"(p));
    } else {
        static_assert(VEC == 8, "vector width");
        asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]) : "l"(p));
    }
}

// keep the slabs n in [lo,hi] on which -1 < A + n*s < N can hold (one slab of slack on each side)
__device__ __forceinline__ void clip_range(double A, double s, int N, double &lo, double &hi)
{
    if (fabs(s) < 1e-12) {
        if (!(A > -1.0 && A < (double)N)) hi = lo - 1.0;
        return;
    }
    double t0 = (-1.0 - A) / s, t1 = ((double)N - A) / s;
    if (t0 > t1) { const double t = t0; t0 = t1; t1 = t; }
    lo = fmax(lo, t0 - 1.0);
    hi = fmin(hi, t1 + 1.0);
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// One slab's four bilinear taps of a ray: offsets from the volume base in float4 units (clamped into the
// volume) and weights (0 for taps outside the volume: zero padding, S8).
struct __align__(16) SlabTaps {
    int o00, o10, o01, o11;
    float w00, w10, w01, w11;
};

// Tile of rays per block: TK rays along k (fastest), RPB/TK along j.
// COOP (VEC == 4 only): the G lanes of a ray take turns at the index arithmetic — lane q works out the taps of
// slab nb+q once, parks them in shared memory, and all lanes then stream through G slabs doing nothing but
// loads and FMAs (v1 spent 21 instructions per LDG.128, profiles/r01_ncu_c5_v1.md).
template <int VEC, int G, int NQ, int DMAX, int MODE, bool COOP, bool LERP = false>
__global__ void __launch_bounds__(256, (COOP && (VEC == 8 || NQ >= 3)) ? FWD_MINB8 : FWD_MINB) john_forward_kernel(const FwdArgs a)
{
    constexpr int RPB = 256 / G;                  // rays per block
    constexpr int TK = (RPB >= 64) ? 8 : (RPB >= 32 ? FWD_TK : (RPB >= 4 ? 4 : RPB));
    constexpr int TJ = RPB / TK;
    const int tid = threadIdx.x;
    const int q = tid % G;                        // lane within the ray's group
    const int r = tid / G;                        // ray within the block
    // MIX (ldk = 48 only): lane q owns channels 8q..8q+7 (one 32-byte load) and 32+4q..32+4q+3 (one 16-byte load),
    // so a warp's request touches each 192-byte record in a 128-byte and a 64-byte piece: 2.5 cache lines per
    // tap on average against 3 for three 64-byte pieces (a load costs one L1 wavefront per distinct line).
    constexpr bool MIX = FWD_MIX48 && VEC == 4 && G == 4 && NQ == 3;
    // LERP (MIX only; the volume is the library's own copy with an all-zero record appended): the bilinear value of a
    // slab is formed as nested differences, c00 + fu (c10 - c00) etc. (scalar fp32; see the march below).  A constant (or slowly
    // varying) field is then reproduced exactly, so a run of slabs through a uniform region adds exact multiples of
    // the voxel value.  Four weighted FMAs make the partial sums of such a run approach powers of two from below,
    // where round-to-nearest is one-sided: a bias of ~-0.2 ulp per slab, coherent over all rays and amplified by A^T
    // (config 5's clipped-ellipsoid density: E_inf(grad) 9e-6 on its own data recipe, nine tenths of it this bias;
    // 1.3e-6 with the nested form).  Taps outside the volume read the zero record, so no 0 x voxel product exists.
    static_assert(!LERP || MIX, "LERP is the ldk = 48 path");
    auto chan = [&](int t) -> int {               // first channel of accumulator vector t of this lane
        if constexpr (MIX) return t < 2 ? 8 * q + 4 * t : 32 + 4 * q;
        else return VEC * (q + G * t);
    };
    const int tiles_k = (a.Kd + TK - 1) / TK, tiles_j = (a.J + TJ - 1) / TJ;
    // Block order: FWD_GS consecutive projections (neighbouring rotation angles) are interleaved tile by tile, so
    // blocks resident at the same time walk the same band of the volume for several projections and the second
    // to FWD_GS-th reader of a voxel finds it in L2 instead of HBM.
    const int tpp = tiles_k * tiles_j;                                   // tiles per projection
    const int grp = blockIdx.x / (FWD_GS * tpp);
    const int rem = blockIdx.x - grp * (FWD_GS * tpp);
    const int gs = min(FWD_GS, a.P - grp * FWD_GS);                      // the last group may be short
    int tile = rem / gs;
    const int s = grp * FWD_GS + rem % gs;
    const int tk = tile % tiles_k; tile /= tiles_k;
    const int tj = tile;
    const int j = tj * TJ + r / TK, k = tk * TK + r % TK;
    const bool ray_ok = (j < a.J) && (k < a.Kd);

    const MMProj *pg = a.tab + s;
    const int m = pg->m, u = pg->u, v = pg->v;
    // (m,u,v) is one of (0,1,2), (1,0,2), (2,0,1)
    const int Nm = (m == 0) ? a.X : (m == 1 ? a.Y : a.Z);
    const int Nu = (u == 0) ? a.X : a.Y, Nv = (v == 2) ? a.Z : a.Y;
    const long long sX = (long long)a.Y * a.Z * a.ldk, sY = (long long)a.Z * a.ldk, sZ = a.ldk;
    const long long sM = (m == 0) ? sX : (m == 1 ? sY : sZ);
    const long long sU = (u == 0) ? sX : sY, sV = (v == 2) ? sZ : sY;

    // Accumulation: fp32 FMAs run over a short round of slabs only (4 taps x U slabs, starting from
    // zero), then the round is added to an fp64 total.  A plain fp32 running sum over <= 256 slabs x 4 taps carries
    // ~3e-7 of the ray sum in rounding, which the residual r = Ac - data (1 % of Ac at 1e4 counts) magnifies to
    // ~3e-5 in the gradient; with short rounds the rounding is relative to the round's own partial sum (~1e-8).
    float acc[NQ][VEC];
    double tot[NQ][VEC];
#pragma unroll
    for (int t = 0; t < NQ; t++)
#pragma unroll
        for (int x = 0; x < VEC; x++) { acc[t][x] = 0.f; tot[t][x] = 0.0; }
    auto flush = [&]() {
#pragma unroll
        for (int t = 0; t < NQ; t++)
#pragma unroll
            for (int x = 0; x < VEC; x++) { tot[t][x] += (double)acc[t][x]; acc[t][x] = 0.f; }
    };

    if constexpr (COOP) {
        static_assert(!COOP || VEC == 4 || VEC == 8, "cooperative march needs 16- or 32-byte lanes");
        // slabs in flight per lane: 32-byte lanes keep a whole round of 8 slabs (32 LDG.256) in flight with 2 blocks
        // per SM (measured best: 210 ms vs 227 ms for 16-byte lanes, 2 slabs, 4 blocks on config 5)
        constexpr int U = (VEC == 8) ? (G < FWD_U8 ? G : FWD_U8) : (NQ >= 3 ? (G < 4 ? G : 4) : FWD_U);
        static_assert(G % U == 0, "a round of G slabs is consumed U at a time");
        // offsets and weights in separate arrays, each ray's row padded by one entry: the rays of a warp then sit in
        // different banks (the [RPB][G] array of 32-byte structs put them all on the same four banks: 9.5 shared
        // wavefronts per warp and slab in profiles/r01_ncu_c5_v4.md, against 3 without conflicts)
        __shared__ int4 tap_o[RPB][G + 1];
        __shared__ float4 tap_w[RPB][G + 1];
        int n0 = 0, n1 = -1;
        long long pu0 = 0, pv0 = 0;
        if (ray_ok) {
            const double Au = pg->Cu + (double)j * pg->Mju + (double)k * pg->Mku;
            const double Av = pg->Cv + (double)j * pg->Mjv + (double)k * pg->Mkv;
            double lo = 0.0, hi = (double)(Nm - 1);
            clip_range(Au, pg->su, Nu, lo, hi);
            clip_range(Av, pg->sv, Nv, lo, hi);
            n0 = (int)ceil(lo); n1 = (int)floor(hi);
            pu0 = (long long)floor(Au * FX_ONE);
            pv0 = (long long)floor(Av * FX_ONE);
        }
        const long long su_fx = pg->su_fx, sv_fx = pg->sv_fx;
        // tap offsets are counted in lane vectors (VEC floats)
        const int ldk4 = a.ldk / VEC;
        const int sM4 = (int)(sM / VEC), sU4 = (int)(sU / VEC), sV4 = (int)(sV / VEC);
        const int zero_off = LERP ? a.zero_vox * ldk4 : 0;
        // All rays of the block start at the block's first slab (slabs before a ray's own n0 carry zero weights):
        // neighbouring rays are then at the SAME slab in the same round and find each other's taps in L1.  With
        // every ray starting at its own n0 they were up to a tile's width of slabs apart (FWD_COMMON_START).
        int nstart = n0;
        if constexpr (FWD_COMMON_START && LERP) {                 // measured on the ldk = 48 path only (config 5: -4 %)
            __shared__ int s_nbeg;
            if (tid == 0) s_nbeg = 0x7fffffff;
            __syncthreads();
            if (q == 0 && n1 >= n0) atomicMin(&s_nbeg, n0);
            __syncthreads();
            nstart = s_nbeg;
        }
        int rounds = (n1 >= n0) ? (n1 - nstart + G) / G : 0;
        rounds = __reduce_max_sync(0xffffffffu, rounds);          // the warp's groups step through rounds together
        for (int rd = 0; rd < rounds; rd++) {
            const int nb = nstart + rd * G;
            {   // lane q: taps of slab nb + q
                const int n = nb + q;
                SlabTaps t;
                t.o00 = t.o10 = t.o01 = t.o11 = 0;
                t.w00 = t.w10 = t.w01 = t.w11 = 0.f;
                if (n >= n0 && n <= n1) {
                    // 24.40 fixed point: the integer part is the tap index, the fraction the bilinear weight
                    const long long pu = pu0 + (long long)n * su_fx, pv = pv0 + (long long)n * sv_fx;
                    const int iu = (int)(pu >> FX_BITS), iv = (int)(pv >> FX_BITS);
                    const float fu = (float)(unsigned int)(pu >> (FX_BITS - 32)) * FX_INV;
                    const float fv = (float)(unsigned int)(pv >> (FX_BITS - 32)) * FX_INV;
                    const bool u0 = (unsigned)iu < (unsigned)Nu, u1 = (unsigned)(iu + 1) < (unsigned)Nu;
                    const bool v0 = (unsigned)iv < (unsigned)Nv, v1 = (unsigned)(iv + 1) < (unsigned)Nv;
                    const int b0 = n * sM4 + (u0 ? iu * sU4 : 0), b1 = n * sM4 + (u1 ? (iu + 1) * sU4 : 0);
                    const int c0 = v0 ? iv * sV4 : 0, c1 = v1 ? (iv + 1) * sV4 : 0;
                    t.o00 = b0 + c0; t.o10 = b1 + c0; t.o01 = b0 + c1; t.o11 = b1 + c1;
                    if constexpr (LERP) {
                        // taps outside the volume read the all-zero record (zero padding, S8); the table carries the fractions
                        if (!(u0 && v0)) t.o00 = zero_off;
                        if (!(u1 && v0)) t.o10 = zero_off;
                        if (!(u0 && v1)) t.o01 = zero_off;
                        if (!(u1 && v1)) t.o11 = zero_off;
                        t.w00 = fu; t.w10 = fv;
                    } else {
                        t.w00 = (u0 && v0) ? (1.f - fu) * (1.f - fv) : 0.f;
                        t.w10 = (u1 && v0) ? fu * (1.f - fv) : 0.f;
                        t.w01 = (u0 && v1) ? (1.f - fu) * fv : 0.f;
                        t.w11 = (u1 && v1) ? fu * fv : 0.f;
                    }
                } else if constexpr (LERP) {
                    t.o00 = t.o10 = t.o01 = t.o11 = zero_off;
                }
                tap_o[r][q] = make_int4(t.o00, t.o10, t.o01, t.o11);
                tap_w[r][q] = make_float4(t.w00, t.w10, t.w01, t.w11);
            }
            __syncwarp();
            // U slabs per step: all their loads are issued before the first FMA (slabs past n1 carry
            // zero weights and offset 0, so the tail needs no special case)
            const int cnt = min(G, n1 - nb + 1);
            for (int i = 0; i < cnt; i += U) {
                int4 o[U];
                float4 w[U];
#pragma unroll
                for (int uu = 0; uu < U; uu++) {
                    o[uu] = tap_o[r][i + uu];
                    w[uu] = tap_w[r][i + uu];
                }
                if constexpr (LERP) {
                    const float *base = a.vol + 8 * q, *base2 = a.vol + 32 + 4 * q;
                    // the round's three load batches (64 registers each): channels 0-31 of slabs 0-1 and of slabs 2-3,
                    // channels 32-47 of all four slabs.  Scalar arithmetic on purpose: the same sub / fma / add sequence
                    // in packed pairs (FADD2 / FFMA2, 42 instead of 84 instructions per lane and slab) is bit-identical
                    // and 5 % SLOWER (config 5: 190.8 against 180.5 ms) — the march waits on latency, not on issue slots,
                    // and the packed chains are longer.
                    float cA[2][4][8], cC[U][4][4];
                    auto load_fh = [&](int hh) {
#pragma unroll
                        for (int uu = 0; uu < 2; uu++) {
                            ldg_nc_vec<8>(base + (long long)o[hh + uu].x * 4, cA[uu][0]);
                            ldg_nc_vec<8>(base + (long long)o[hh + uu].y * 4, cA[uu][1]);
                            ldg_nc_vec<8>(base + (long long)o[hh + uu].z * 4, cA[uu][2]);
                            ldg_nc_vec<8>(base + (long long)o[hh + uu].w * 4, cA[uu][3]);
                        }
                    };
                    auto math_fh = [&](int hh) {
#pragma unroll
                        for (int uu = 0; uu < 2; uu++) {
                            const float fu = w[hh + uu].x, fv = w[hh + uu].y;
#pragma unroll
                            for (int x = 0; x < 8; x++) {
                                const float t0 = fmaf(fu, cA[uu][1][x] - cA[uu][0][x], cA[uu][0][x]);
                                const float t1 = fmaf(fu, cA[uu][3][x] - cA[uu][2][x], cA[uu][2][x]);
                                acc[x / 4][x % 4] += fmaf(fv, t1 - t0, t0);
                            }
                        }
                    };
                    auto load_up = [&]() {
#pragma unroll
                        for (int uu = 0; uu < U; uu++) {
                            ldg_nc_vec<4>(base2 + (long long)o[uu].x * 4, cC[uu][0]);
                            ldg_nc_vec<4>(base2 + (long long)o[uu].y * 4, cC[uu][1]);
                            ldg_nc_vec<4>(base2 + (long long)o[uu].z * 4, cC[uu][2]);
                            ldg_nc_vec<4>(base2 + (long long)o[uu].w * 4, cC[uu][3]);
                        }
                    };
                    auto math_up = [&]() {
#pragma unroll
                        for (int uu = 0; uu < U; uu++) {
                            const float fu = w[uu].x, fv = w[uu].y;
#pragma unroll
                            for (int x = 0; x < 4; x++) {
                                const float t0 = fmaf(fu, cC[uu][1][x] - cC[uu][0][x], cC[uu][0][x]);
                                const float t1 = fmaf(fu, cC[uu][3][x] - cC[uu][2][x], cC[uu][2][x]);
                                acc[2][x] += fmaf(fv, t1 - t0, t0);
                            }
                        }
                    };
                    static_assert(U == 4, "the nested-difference march consumes rounds of four slabs");
                    load_fh(0);
                    flush();                                      // the previous round's sums, under this round's load latency
                    math_fh(0);
                    load_fh(2); math_fh(2);
                    load_up(); math_up();
                } else if constexpr (MIX) {
                    const float *base = a.vol + 8 * q, *base2 = a.vol + 32 + 4 * q;
#pragma unroll
                    for (int h = 0; h < U; h += 2) {              // 32-byte pieces, two slabs at a time
                        float c[2][4][8];
#pragma unroll
                        for (int uu = 0; uu < 2; uu++) {
                            ldg_nc_vec<8>(base + (long long)o[h + uu].x * 4, c[uu][0]);
                            ldg_nc_vec<8>(base + (long long)o[h + uu].y * 4, c[uu][1]);
                            ldg_nc_vec<8>(base + (long long)o[h + uu].z * 4, c[uu][2]);
                            ldg_nc_vec<8>(base + (long long)o[h + uu].w * 4, c[uu][3]);
                        }
                        if (h == 0) flush();                      // the previous step's sums, under this step's load latency
#pragma unroll
                        for (int uu = 0; uu < 2; uu++) {
                            const float ww[4] = {w[h + uu].x, w[h + uu].y, w[h + uu].z, w[h + uu].w};
#pragma unroll
                            for (int p = 0; p < 4; p++)
#pragma unroll
                                for (int x = 0; x < 8; x++) acc[x / 4][x % 4] = fmaf(ww[p], c[uu][p][x], acc[x / 4][x % 4]);
                        }
                    }
                    float c[U][4][4];                             // 16-byte pieces
#pragma unroll
                    for (int uu = 0; uu < U; uu++) {
                        ldg_nc_vec<4>(base2 + (long long)o[uu].x * 4, c[uu][0]);
                        ldg_nc_vec<4>(base2 + (long long)o[uu].y * 4, c[uu][1]);
                        ldg_nc_vec<4>(base2 + (long long)o[uu].z * 4, c[uu][2]);
                        ldg_nc_vec<4>(base2 + (long long)o[uu].w * 4, c[uu][3]);
                    }
#pragma unroll
                    for (int uu = 0; uu < U; uu++) {
                        const float ww[4] = {w[uu].x, w[uu].y, w[uu].z, w[uu].w};
#pragma unroll
                        for (int p = 0; p < 4; p++)
#pragma unroll
                            for (int x = 0; x < 4; x++) acc[2][x] = fmaf(ww[p], c[uu][p][x], acc[2][x]);
                    }
                } else {
    #pragma unroll
                    for (int t = 0; t < NQ; t++) {
                        // lanes past the last float4 of the voxel re-read its last one (same cache line, result
                        // discarded in the epilogue): no branch in the loop
                        const int e = min(q + G * t, ldk4 - 1);
                        float c[U][4][VEC];
    #pragma unroll
                        for (int uu = 0; uu < U; uu++) {
                            ldg_nc_vec<VEC>(a.vol + (long long)(o[uu].x + e) * VEC, c[uu][0]);
                            ldg_nc_vec<VEC>(a.vol + (long long)(o[uu].y + e) * VEC, c[uu][1]);
                            ldg_nc_vec<VEC>(a.vol + (long long)(o[uu].z + e) * VEC, c[uu][2]);
                            ldg_nc_vec<VEC>(a.vol + (long long)(o[uu].w + e) * VEC, c[uu][3]);
                        }
                        if (t == 0) flush();                      // the previous step's sums, under this step's load latency
    #pragma unroll
                        for (int uu = 0; uu < U; uu++) {
                            const float ww[4] = {w[uu].x, w[uu].y, w[uu].z, w[uu].w};
    #pragma unroll
                            for (int p = 0; p < 4; p++)
    #pragma unroll
                                for (int x = 0; x < VEC; x++) acc[t][x] = fmaf(ww[p], c[uu][p][x], acc[t][x]);
                        }
                    }
                }
            }
            __syncwarp();
        }
        flush();
    } else if (ray_ok) {
        const double Au = pg->Cu + (double)j * pg->Mju + (double)k * pg->Mku;
        const double Av = pg->Cv + (double)j * pg->Mjv + (double)k * pg->Mkv;
        double lo = 0.0, hi = (double)(Nm - 1);
        clip_range(Au, pg->su, Nu, lo, hi);
        clip_range(Av, pg->sv, Nv, lo, hi);
        const int n0 = (int)ceil(lo), n1 = (int)floor(hi);
        const long long su_fx = pg->su_fx, sv_fx = pg->sv_fx;
        // 24.40 fixed point: the integer part is the tap index, the fraction the bilinear weight
        long long pu = (long long)floor(Au * FX_ONE) + (long long)n0 * su_fx;
        long long pv = (long long)floor(Av * FX_ONE) + (long long)n0 * sv_fx;
        const float *slab = a.vol + (long long)n0 * sM;
        for (int n = n0; n <= n1; n++) {
            const int iu = (int)(pu >> FX_BITS), iv = (int)(pv >> FX_BITS);
            const float fu = (float)(unsigned int)(pu >> (FX_BITS - 32)) * FX_INV;
            const float fv = (float)(unsigned int)(pv >> (FX_BITS - 32)) * FX_INV;
            const bool u0 = (unsigned)iu < (unsigned)Nu, u1 = (unsigned)(iu + 1) < (unsigned)Nu;
            const bool v0 = (unsigned)iv < (unsigned)Nv, v1 = (unsigned)(iv + 1) < (unsigned)Nv;
            const float w00 = (1.f - fu) * (1.f - fv), w10 = fu * (1.f - fv), w01 = (1.f - fu) * fv, w11 = fu * fv;
            const float *p00 = slab + (long long)iu * sU + (long long)iv * sV;
#pragma unroll
            for (int t = 0; t < NQ; t++) {
                const int ch = chan(t);
                if (ch < a.ldk) {
                    float c00[VEC], c10[VEC], c01[VEC], c11[VEC];
#pragma unroll
                    for (int x = 0; x < VEC; x++) c00[x] = c10[x] = c01[x] = c11[x] = 0.f;
                    const float *pe = p00 + ch;
                    if (u0 && v0) Ld<VEC>::ld(pe, c00);
                    if (u1 && v0) Ld<VEC>::ld(pe + sU, c10);
                    if (u0 && v1) Ld<VEC>::ld(pe + sV, c01);
                    if (u1 && v1) Ld<VEC>::ld(pe + sU + sV, c11);
#pragma unroll
                    for (int x = 0; x < VEC; x++) {
                        acc[t][x] = fmaf(w00, c00[x], acc[t][x]);
                        acc[t][x] = fmaf(w10, c10[x], acc[t][x]);
                        acc[t][x] = fmaf(w01, c01[x], acc[t][x]);
                        acc[t][x] = fmaf(w11, c11[x], acc[t][x]);
                    }
                }
            }
            pu += su_fx; pv += sv_fx; slab += sM;
            if (((n - n0) & 7) == 7) flush();
        }
        flush();
    }
    const double w = pg->w64;                     // Joseph step a/|d_m| in fp64: its fp32 rounding is a per-projection scale error
    const long long ray = ((long long)s * a.J + j) * a.Kd + k;

    if constexpr (MODE == 0) {
        if (!ray_ok) return;
#pragma unroll
        for (int t = 0; t < NQ; t++) {
            const int ch = chan(t);
            if (ch < a.ldk) {
                float o[VEC];
#pragma unroll
                for (int x = 0; x < VEC; x++) o[x] = (ch + x < a.K) ? (float)(w * tot[t][x]) : 0.f;
                Ld<VEC>::st(a.proj + ray * a.ldk + ch, o);
            }
        }
        return;
    } else {

    // fused reciprocal-space map (Eq. 6): Imod[c] = sum_i B[s][i][c] p[i], reduced over the ray's G lanes
    // in fp64: 45 x 8 DFMA per ray, once per ray — nothing next to the march, and the residual below is then
    // formed from an unrounded model value
    double part[DMAX];
#pragma unroll
    for (int c = 0; c < DMAX; c++) part[c] = 0.0;
    const float *Bs = a.B + (long long)s * a.K * a.D;
#pragma unroll
    for (int t = 0; t < NQ; t++) {
        const int ch = chan(t);
#pragma unroll
        for (int x = 0; x < VEC; x++) {
            const int i = ch + x;
            if (i < a.K) {
                const double pv_ = w * tot[t][x];
#pragma unroll
                for (int c = 0; c < DMAX; c++)
                    if (c < a.D) part[c] = fma((double)__ldg(Bs + (long long)i * a.D + c), pv_, part[c]);
            }
        }
    }
    if constexpr (G > 1) {
#pragma unroll
        for (int o = G / 2; o > 0; o >>= 1)
#pragma unroll
            for (int c = 0; c < DMAX; c++) part[c] += __shfl_xor_sync(0xffffffffu, part[c], o);
    }

    double lsum = 0.0;
#pragma unroll
    for (int c = 0; c < DMAX; c++) {
        if ((c % G) == q && c < a.D && ray_ok) {
            const long long o = ray * a.D + c;
            if (MODE == 1) {
                a.sino[o] = (float)part[c];
            } else {
                const double res = part[c] - (double)__ldg(a.data + o);   // r = Ac - I  (Eq. 13), unrounded model value
                const double wt = a.weights ? (double)__ldg(a.weights + o) : 1.0;
                double psi = res;                                          // rho'(r): r, or clip(r, -delta, delta) (Huber, S23)
                double rho = 0.5 * res * res;                              // L = sum w rho(r): 1/2 r^2 (S10) ...
                if (a.huber > 0.f && fabs(res) > (double)a.huber) {
                    psi = copysign((double)a.huber, res);
                    rho = (double)a.huber * (fabs(res) - 0.5 * (double)a.huber);   // ... or delta (|r| - delta/2)
                }
                a.sino[o] = (float)(wt * psi);
                lsum += wt * rho;
            }
        }
    }
    if (MODE == 2) {
        __shared__ double red[8];
        lsum = warp_sum(lsum);
        if ((tid & 31) == 0) red[tid >> 5] = lsum;
        __syncthreads();
        if (tid == 0) {
            double tot = 0.0;
#pragma unroll
            for (int i = 0; i < 8; i++) tot += red[i];
            if (tot != 0.0) atomicAdd(a.loss, tot);
        }
    }
    }   // MODE != 0
}

// ================================================================================================
// adjoint, K-channel (standalone mm_john_adjoint): voxel-stationary gather, lanes over channels
// ================================================================================================
template <int VEC, int G, int NQ>
__global__ void __launch_bounds__(256) john_adjoint_kernel(const AdjArgs a)
{
    constexpr int VPB = 256 / G;
    const int tid = threadIdx.x;
    const int q = tid % G;
    const long long vox = (long long)blockIdx.x * VPB + tid / G;
    const long long nvox = (long long)a.X * a.Y * a.Z;
    if (vox >= nvox) return;
    const int z = (int)(vox % a.Z), y = (int)((vox / a.Z) % a.Y), x = (int)(vox / ((long long)a.Z * a.Y));
    float acc[NQ][VEC];
#pragma unroll
    for (int t = 0; t < NQ; t++)
#pragma unroll
        for (int c = 0; c < VEC; c++) acc[t][c] = 0.f;

    for (int s = 0; s < a.P; s++) {
        const MMProj *pg = a.tab + s;
        const double j0 = fma((double)x, pg->Jx[0], fma((double)y, pg->Jx[1], fma((double)z, pg->Jx[2], pg->Jc)));
        const double k0 = fma((double)x, pg->Kx[0], fma((double)y, pg->Kx[1], fma((double)z, pg->Kx[2], pg->Kc)));
        const double fj0 = floor(j0), fk0 = floor(k0);
        const int jb = (int)fj0, kb = (int)fk0;
        const float fj = (float)(j0 - fj0), fk = (float)(k0 - fk0);
        const float hj = pg->hj, hk = pg->hk, w = pg->w;
        const float mju = pg->mju, mku = pg->mku, mjv = pg->mjv, mkv = pg->mkv;
        // bilinear mode: the four pixels around (j0,k0) with weights (1-fj | fj)(1-fk | fk)
        const int djlo = max(a.bilinear ? 0 : (int)ceilf(fj - hj), -jb), djhi = min(a.bilinear ? 1 : (int)floorf(fj + hj), a.J - 1 - jb);
        const int dklo = max(a.bilinear ? 0 : (int)ceilf(fk - hk), -kb), dkhi = min(a.bilinear ? 1 : (int)floorf(fk + hk), a.Kd - 1 - kb);
        for (int dj = djlo; dj <= djhi; dj++) {
            const float ej = (float)dj - fj;
            for (int dk = dklo; dk <= dkhi; dk++) {
                const float ek = (float)dk - fk;
                const float du = a.bilinear ? ej : fmaf(mju, ej, mku * ek), dv = a.bilinear ? ek : fmaf(mjv, ej, mkv * ek);
                const float wt = w * fmaxf(0.f, 1.f - fabsf(du)) * fmaxf(0.f, 1.f - fabsf(dv));
                if (wt > 0.f) {
                    const float *p = a.src + (((long long)s * a.J + (jb + dj)) * a.Kd + (kb + dk)) * a.ldk;
#pragma unroll
                    for (int t = 0; t < NQ; t++) {
                        const int e = q + G * t;
                        if (VEC * e < a.ldk) {
                            float c[VEC];
                            Ld<VEC>::ld(p + VEC * e, c);
#pragma unroll
                            for (int xx = 0; xx < VEC; xx++) acc[t][xx] = fmaf(wt, c[xx], acc[t][xx]);
                        }
                    }
                }
            }
        }
    }
#pragma unroll
    for (int t = 0; t < NQ; t++) {
        const int e = q + G * t;
        if (VEC * e < a.ldk) {
            float o[VEC];
#pragma unroll
            for (int xx = 0; xx < VEC; xx++) o[xx] = (VEC * e + xx < a.K) ? acc[t][xx] : 0.f;
            Ld<VEC>::st(a.out + vox * a.ldk + VEC * e, o);
        }
    }
}

// ================================================================================================
// adjoint, fused (mm_adjoint, phase 2 of mm_loss_gradient): thread per voxel gathers the D-channel
// sinogram with the exact-transpose weights, then applies B_s^T; K accumulators live in registers.
// ================================================================================================
#define ADJ_PCH 8        // projections staged in shared memory per step

struct AdjProjS {        // the fields of MMProj the gather needs
    double Jc, Jx0, Jx1, Jx2, Kc, Kx0, Kx1, Kx2;
    float mju, mku, mjv, mkv, hj, hk, w, pad;
};

template <int KMAX, int DMAX>
__global__ void __launch_bounds__(128) adjoint_fused_kernel(const AdjArgs a)
{
    __shared__ AdjProjS sp[ADJ_PCH];
    __shared__ __align__(16) float sB[ADJ_PCH][KMAX * DMAX];
    const int tid = threadIdx.x;
    const long long vox = a.vox_begin + (long long)blockIdx.x * 128 + tid;
    const long long nvox = a.vox_end;
    const bool ok = vox < nvox;
    const long long vv = ok ? vox : nvox - 1;
    const int z = (int)(vv % a.Z), y = (int)((vv / a.Z) % a.Y), x = (int)(vv / ((long long)a.Z * a.Y));
    const int i0 = blockIdx.y * KMAX;             // channel chunk handled by this block
    float acc[KMAX];
#pragma unroll
    for (int i = 0; i < KMAX; i++) acc[i] = 0.f;

    for (int s0 = 0; s0 < a.P; s0 += ADJ_PCH) {
        const int ns = min(ADJ_PCH, a.P - s0);
        __syncthreads();
        if (tid < ns) {
            const MMProj *pg = a.tab + s0 + tid;
            AdjProjS t;
            t.Jc = pg->Jc; t.Jx0 = pg->Jx[0]; t.Jx1 = pg->Jx[1]; t.Jx2 = pg->Jx[2];
            t.Kc = pg->Kc; t.Kx0 = pg->Kx[0]; t.Kx1 = pg->Kx[1]; t.Kx2 = pg->Kx[2];
            t.mju = pg->mju; t.mku = pg->mku; t.mjv = pg->mjv; t.mkv = pg->mkv;
            t.hj = pg->hj; t.hk = pg->hk; t.w = pg->w; t.pad = 0.f;
            sp[tid] = t;
        }
        for (int idx = tid; idx < ns * KMAX * DMAX; idx += 128) {
            const int ps = idx / (KMAX * DMAX), rem = idx % (KMAX * DMAX);
            const int i = i0 + rem / DMAX, c = rem % DMAX;
            sB[ps][rem] = (i < a.K && c < a.D) ? __ldg(a.B + ((long long)(s0 + ps) * a.K + i) * a.D + c) : 0.f;
        }
        __syncthreads();
        for (int ps = 0; ps < ns; ps++) {
            const AdjProjS &pg = sp[ps];
            const int s = s0 + ps;
            float t[DMAX];
#pragma unroll
            for (int c = 0; c < DMAX; c++) t[c] = 0.f;
            const double j0 = fma((double)x, pg.Jx0, fma((double)y, pg.Jx1, fma((double)z, pg.Jx2, pg.Jc)));
            const double k0 = fma((double)x, pg.Kx0, fma((double)y, pg.Kx1, fma((double)z, pg.Kx2, pg.Kc)));
            const double fj0 = floor(j0), fk0 = floor(k0);
            const int jb = (int)fj0, kb = (int)fk0;
            const float fj = (float)(j0 - fj0), fk = (float)(k0 - fk0);
            const int djlo = max(a.bilinear ? 0 : (int)ceilf(fj - pg.hj), -jb), djhi = min(a.bilinear ? 1 : (int)floorf(fj + pg.hj), a.J - 1 - jb);
            const int dklo = max(a.bilinear ? 0 : (int)ceilf(fk - pg.hk), -kb), dkhi = min(a.bilinear ? 1 : (int)floorf(fk + pg.hk), a.Kd - 1 - kb);
            for (int dj = djlo; dj <= djhi; dj++) {
                const float ej = (float)dj - fj;
                for (int dk = dklo; dk <= dkhi; dk++) {
                    const float ek = (float)dk - fk;
                    const float du = a.bilinear ? ej : fmaf(pg.mju, ej, pg.mku * ek), dv = a.bilinear ? ek : fmaf(pg.mjv, ej, pg.mkv * ek);
                    const float wt = pg.w * fmaxf(0.f, 1.f - fabsf(du)) * fmaxf(0.f, 1.f - fabsf(dv));
                    if (wt > 0.f) {
                        const float *p = a.src + (((long long)s * a.J + (jb + dj)) * a.Kd + (kb + dk)) * a.D;
                        if (a.vec_ok) {
#pragma unroll
                            for (int c = 0; c < DMAX; c += 4) {
                                if (c < a.D) {
                                    const float4 r = __ldg(reinterpret_cast<const float4 *>(p + c));
                                    t[c] = fmaf(wt, r.x, t[c]); t[c + 1] = fmaf(wt, r.y, t[c + 1]);
                                    t[c + 2] = fmaf(wt, r.z, t[c + 2]); t[c + 3] = fmaf(wt, r.w, t[c + 3]);
                                }
                            }
                        } else {
#pragma unroll
                            for (int c = 0; c < DMAX; c++)
                                if (c < a.D) t[c] = fmaf(wt, __ldg(p + c), t[c]);
                        }
                    }
                }
            }
            // acc[i] += sum_c B[s][i][c] t[c]   (transpose of Eq. 6's inner sum)
            const float4 *b4 = reinterpret_cast<const float4 *>(sB[ps]);
#pragma unroll
            for (int i = 0; i < KMAX; i++) {
#pragma unroll
                for (int c = 0; c < DMAX; c += 4) {
                    const float4 b = b4[(i * DMAX + c) / 4];
                    acc[i] = fmaf(b.x, t[c], acc[i]); acc[i] = fmaf(b.y, t[c + 1], acc[i]);
                    acc[i] = fmaf(b.z, t[c + 2], acc[i]); acc[i] = fmaf(b.w, t[c + 3], acc[i]);
                }
            }
        }
    }
    if (!ok) return;
    float *o = a.out + vox * a.ldk;
#pragma unroll
    for (int i = 0; i < KMAX; i++) {
        const int ch = i0 + i;
        if (ch < a.ldk) o[ch] = (ch < a.K) ? acc[i] : 0.f;
    }
}

// ================================================================================================
// standalone reciprocal-space maps and the GD update
// ================================================================================================
__global__ void basis_forward_kernel(const float *__restrict__ B, const float *__restrict__ proj, float *__restrict__ sino,
                                     int K, int ldk, int D, long long npix_per_proj, long long total)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // (pixel, c)
    if (idx >= total) return;
    const long long pix = idx / D;
    const int c = (int)(idx % D);
    const long long s = pix / npix_per_proj;
    const float *Bs = B + s * K * D + c;
    const float *p = proj + pix * ldk;
    float sum = 0.f;
    for (int i = 0; i < K; i++) sum = fmaf(__ldg(Bs + (long long)i * D), __ldg(p + i), sum);
    sino[idx] = sum;
}

__global__ void basis_adjoint_kernel(const float *__restrict__ B, const float *__restrict__ sino, float *__restrict__ proj,
                                     int K, int ldk, int D, long long npix_per_proj, long long total)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // (pixel, i)
    if (idx >= total) return;
    const long long pix = idx / ldk;
    const int i = (int)(idx % ldk);
    float sum = 0.f;
    if (i < K) {
        const long long s = pix / npix_per_proj;
        const float *Bs = B + (s * K + i) * D;
        const float *y = sino + pix * D;
        for (int c = 0; c < D; c++) sum = fmaf(__ldg(Bs + c), __ldg(y + c), sum);
    }
    proj[idx] = sum;
}

__global__ void axpy_kernel(float *__restrict__ c, const float *__restrict__ g, float eta, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) c[i] = fmaf(-eta, g[i], c[i]);
}

// SIRT/MITRA: x <- 1/x where x > floor, else 0 (rays that miss the sample, unseen voxels)
__global__ void reciprocal_kernel(float *__restrict__ x, float floor_, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { const float v = x[i]; x[i] = v > floor_ ? 1.f / v : 0.f; }
}

// NEXT-3: zero-padded 7-point Laplacian of every channel; one thread per float4 of the volume,
// neighbours along z are adjacent records, along y and x one row / plane away (all coalesced 16-byte loads)
template <int VEC>
__global__ void laplacian_kernel(const float *__restrict__ in, float *__restrict__ out, int X, int Y, int Z, int ldk, int K)
{
    const int lpv = ldk / VEC;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)X * Y * Z * lpv;
    if (idx >= total) return;
    const int e = (int)(idx % lpv);
    const long long vox = idx / lpv;
    const int z = (int)(vox % Z), y = (int)((vox / Z) % Y), x = (int)(vox / ((long long)Z * Y));
    const long long sZ = ldk, sY = (long long)Z * ldk, sX = (long long)Y * Z * ldk;
    const float *p = in + vox * ldk + VEC * e;
    float c[VEC], acc[VEC], nb[VEC];
    Ld<VEC>::ld(p, c);
#pragma unroll
    for (int i = 0; i < VEC; i++) acc[i] = -6.f * c[i];
#define MM_LAP_TAP(cond, off)                                    \
    if (cond) {                                                  \
        Ld<VEC>::ld(p + (off), nb);                              \
        _Pragma("unroll") for (int i = 0; i < VEC; i++) acc[i] += nb[i]; \
    }
    MM_LAP_TAP(z > 0, -sZ) MM_LAP_TAP(z + 1 < Z, sZ)
    MM_LAP_TAP(y > 0, -sY) MM_LAP_TAP(y + 1 < Y, sY)
    MM_LAP_TAP(x > 0, -sX) MM_LAP_TAP(x + 1 < X, sX)
#undef MM_LAP_TAP
#pragma unroll
    for (int i = 0; i < VEC; i++) acc[i] = (VEC * e + i < K) ? acc[i] : 0.f;
    Ld<VEC>::st(out + vox * ldk + VEC * e, acc);
}

// NEXT-4, derived quantities of an SH coefficient volume (Eq. 10-12), one thread per voxel.
// With 4pi-normalised real harmonics (S14) only l = 0 and l = 2 enter: mean = c_00 and, from <x^2> = 1/3,
// <x^4> = 1/5, <x^2 y^2> = 1/15 and Y_2,-2..2 = sqrt15 xy, sqrt15 yz, (sqrt5/2)(3z^2-1), sqrt15 xz, (sqrt15/2)(x^2-y^2):
//   M_xy = c_1/sqrt15, M_yz = c_2/sqrt15, M_xz = c_4/sqrt15,
//   M_xx = c_0/3 - c_3/(3 sqrt5) + c_5/sqrt15, M_yy = c_0/3 - c_3/(3 sqrt5) - c_5/sqrt15, M_zz = c_0/3 + 2 c_3/(3 sqrt5).
// Eigenvalues of the symmetric 3x3 by the trigonometric formula, eigenvectors from cross products of the rows of
// M - lambda I; all in fp64 (a few hundred flops per voxel against 24..192 bytes of traffic).
__device__ __forceinline__ void eigvec3(const double M[6], double lam, double v[3], double *quality)
{
    // rows of A = M - lam I; the eigenvector is orthogonal to all of them: take the largest cross product
    const double r0[3] = {M[0] - lam, M[3], M[4]}, r1[3] = {M[3], M[1] - lam, M[5]}, r2[3] = {M[4], M[5], M[2] - lam};
    double c[3][3] = {{r0[1] * r1[2] - r0[2] * r1[1], r0[2] * r1[0] - r0[0] * r1[2], r0[0] * r1[1] - r0[1] * r1[0]},
                      {r0[1] * r2[2] - r0[2] * r2[1], r0[2] * r2[0] - r0[0] * r2[2], r0[0] * r2[1] - r0[1] * r2[0]},
                      {r1[1] * r2[2] - r1[2] * r2[1], r1[2] * r2[0] - r1[0] * r2[2], r1[0] * r2[1] - r1[1] * r2[0]}};
    int best = 0;
    double bn = -1.0;
    for (int i = 0; i < 3; i++) {
        const double n = c[i][0] * c[i][0] + c[i][1] * c[i][1] + c[i][2] * c[i][2];
        if (n > bn) { bn = n; best = i; }
    }
    *quality = bn;                                                       // ~ (gap to the other eigenvalues)^4: 0 when lam is repeated
    if (bn > 0.0) { const double s = rsqrt(bn); v[0] = c[best][0] * s; v[1] = c[best][1] * s; v[2] = c[best][2] * s; }
    else { v[0] = 1.0; v[1] = 0.0; v[2] = 0.0; }
}

// Orthonormal eigenvectors of the symmetric M for eigenvalues l[0] >= l[1] >= l[2].  The vector of the best-isolated
// eigenvalue comes from eigvec3; when two eigenvalues (nearly) coincide the other two are ANY orthonormal pair of the
// orthogonal plane (a valid eigenbasis of the repeated eigenvalue), completed by Gram-Schmidt; M = lambda I gives the
// identity frame.  `tiny` = the scale below which a gap counts as zero.
__device__ __forceinline__ void eigframe3(const double M[6], const double l[3], double tiny, double V[3][3])
{
    const double g01 = l[0] - l[1], g12 = l[1] - l[2];
    if (g01 <= tiny && g12 <= tiny) {                                    // isotropic
        for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) V[i][j] = i == j ? 1.0 : 0.0;
        return;
    }
    double q;
    const int iso = g01 >= g12 ? 0 : 2;                                  // the eigenvalue farthest from the other two
    eigvec3(M, l[iso], V[iso], &q);
    const int other = 2 - iso;                                           // 2 or 0; the middle one is index 1
    double qo;
    eigvec3(M, l[other], V[other], &qo);
    const double gap_mid = iso == 0 ? g12 : g01;
    // project the isolated vector out and renormalise; fall back to a coordinate axis in the plane when the pair is repeated
    double d = V[other][0] * V[iso][0] + V[other][1] * V[iso][1] + V[other][2] * V[iso][2];
    double w[3] = {V[other][0] - d * V[iso][0], V[other][1] - d * V[iso][1], V[other][2] - d * V[iso][2]};
    double n = w[0] * w[0] + w[1] * w[1] + w[2] * w[2];
    if (gap_mid <= tiny || n < 0.25) {
        // repeated pair: any unit vector orthogonal to V[iso]; start from the coordinate axis least aligned with it
        const double ax = fabs(V[iso][0]), ay = fabs(V[iso][1]), az = fabs(V[iso][2]);
        double e[3] = {0.0, 0.0, 0.0};
        e[(ax <= ay && ax <= az) ? 0 : (ay <= az ? 1 : 2)] = 1.0;
        d = e[0] * V[iso][0] + e[1] * V[iso][1] + e[2] * V[iso][2];
        w[0] = e[0] - d * V[iso][0]; w[1] = e[1] - d * V[iso][1]; w[2] = e[2] - d * V[iso][2];
        n = w[0] * w[0] + w[1] * w[1] + w[2] * w[2];
    }
    const double s = rsqrt(n);
    V[other][0] = w[0] * s; V[other][1] = w[1] * s; V[other][2] = w[2] * s;
    // the middle vector completes the right-handed frame: iso x other (or other x iso)
    const double *a = V[iso], *b = V[other];
    V[1][0] = a[1] * b[2] - a[2] * b[1]; V[1][1] = a[2] * b[0] - a[0] * b[2]; V[1][2] = a[0] * b[1] - a[1] * b[0];
}

__global__ void derived_kernel(const float *__restrict__ vol, int ldk, int K, long long nvox, float *__restrict__ mean,
                               float *__restrict__ moments, float *__restrict__ eig, float *__restrict__ vec, float *__restrict__ fa)
{
    const long long vox = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (vox >= nvox) return;
    const float *c = vol + vox * ldk;
    const double c0 = c[0];
    double c1 = 0, c2 = 0, c3 = 0, c4 = 0, c5 = 0;
    if (K >= 6) { c1 = c[1]; c2 = c[2]; c3 = c[3]; c4 = c[4]; c5 = c[5]; }
    const double i15 = 0.2581988897471611, i35 = 0.14907119849998599;   // 1/sqrt15, 1/(3 sqrt5)
    double M[6] = {c0 / 3 - c3 * i35 + c5 * i15, c0 / 3 - c3 * i35 - c5 * i15, c0 / 3 + 2 * c3 * i35, c1 * i15, c4 * i15, c2 * i15};
    const double q = (M[0] + M[1] + M[2]) / 3.0;
    const double p1 = M[3] * M[3] + M[4] * M[4] + M[5] * M[5];
    const double d0 = M[0] - q, d1 = M[1] - q, d2 = M[2] - q;
    const double p = sqrt((d0 * d0 + d1 * d1 + d2 * d2 + 2.0 * p1) / 6.0);
    double l[3] = {q, q, q};
    if (p > 0.0) {
        const double b0 = d0 / p, b1 = d1 / p, b2 = d2 / p, b3 = M[3] / p, b4 = M[4] / p, b5 = M[5] / p;
        double r = 0.5 * (b0 * (b1 * b2 - b5 * b5) - b3 * (b3 * b2 - b5 * b4) + b4 * (b3 * b5 - b1 * b4));
        r = fmin(1.0, fmax(-1.0, r));
        const double phi = acos(r) / 3.0;
        l[0] = q + 2.0 * p * cos(phi);
        l[2] = q + 2.0 * p * cos(phi + 2.0943951023931953);
        l[1] = 3.0 * q - l[0] - l[2];
    }
    if (mean) mean[vox] = (float)c0;                                    // Eq. 10: Y_00 = 1
    if (moments) { for (int i = 0; i < 6; i++) moments[vox * 6 + i] = (float)M[i]; }   // xx, yy, zz, xy, xz, yz  (Eq. 11)
    if (eig) { eig[vox * 3] = (float)l[0]; eig[vox * 3 + 1] = (float)l[1]; eig[vox * 3 + 2] = (float)l[2]; }
    if (vec) {
        double V[3][3];
        eigframe3(M, l, 1e-12 * fmax(fabs(l[0]), fabs(l[2])), V);
        for (int i = 0; i < 3; i++) {
            vec[vox * 9 + 3 * i] = (float)V[i][0]; vec[vox * 9 + 3 * i + 1] = (float)V[i][1]; vec[vox * 9 + 3 * i + 2] = (float)V[i][2];
        }
    }
    if (fa) {                                                           // Eq. 12
        const double num = sqrt((l[0] - l[1]) * (l[0] - l[1]) + (l[1] - l[2]) * (l[1] - l[2]) + (l[2] - l[0]) * (l[2] - l[0]));
        const double den = sqrt(2.0 * (l[0] * l[0] + l[1] * l[1] + l[2] * l[2]));
        fa[vox] = den > 0.0 ? (float)(num / den) : 0.f;
    }
}

// NEXT-3 regularisers (reading S24), one thread per (voxel, channel): value (fp64, one atomic per
// block) and gradient.  kind 1: L1Norm, 2: HuberNorm, 3: TotalVariation (Huber norm of the forward-difference
// gradient per channel).  h(t) = t^2/(2 delta) for |t| <= delta, |t| - delta/2 beyond.
__device__ __forceinline__ float reg_huber(float t, float delta)
{
    const float a = fabsf(t);
    return a <= delta ? t * t / (2.f * delta) : a - 0.5f * delta;
}
// forward differences of channel i at voxel (x,y,z) (0 across the last face) and their Euclidean norm
__device__ __forceinline__ float tv_diffs(const float *__restrict__ v, int x, int y, int z, int X, int Y, int Z, long long sX,
                                          long long sY, long long sZ, float (&d)[3])
{
    const float *p = v + x * sX + y * sY + z * sZ;
    const float c = __ldg(p);
    d[0] = x + 1 < X ? __ldg(p + sX) - c : 0.f;
    d[1] = y + 1 < Y ? __ldg(p + sY) - c : 0.f;
    d[2] = z + 1 < Z ? __ldg(p + sZ) - c : 0.f;
    return sqrtf(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
}
__global__ void __launch_bounds__(256) regulariser_kernel(const float *__restrict__ vol, float *__restrict__ grad, double *__restrict__ value,
                                                          int kind, float delta, int X, int Y, int Z, int ldk, int K)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)X * Y * Z * ldk;
    double r = 0.0;
    if (idx < total) {
        const int i = (int)(idx % ldk);
        const long long vox = idx / ldk;
        float g = 0.f;
        if (i < K) {
            const float c = __ldg(vol + idx);
            if (kind == 1) { r = fabsf(c); g = c > 0.f ? 1.f : (c < 0.f ? -1.f : 0.f); }
            else if (kind == 2) { r = reg_huber(c, delta); g = fminf(1.f, fmaxf(-1.f, c / delta)); }
            else {
                const int z = (int)(vox % Z), y = (int)((vox / Z) % Y), x = (int)(vox / ((long long)Z * Y));
                const long long sZ = ldk, sY = (long long)Z * ldk, sX = (long long)Y * Z * ldk;
                const float *v = vol + i;
                float d[3], dn[3];
                const float n = tv_diffs(v, x, y, z, X, Y, Z, sX, sY, sZ, d);
                r = reg_huber(n, delta);
                g = -(d[0] + d[1] + d[2]) / fmaxf(n, delta);                         // - sum_a p_a(x)
                if (x > 0) { const float m = tv_diffs(v, x - 1, y, z, X, Y, Z, sX, sY, sZ, dn); g += dn[0] / fmaxf(m, delta); }
                if (y > 0) { const float m = tv_diffs(v, x, y - 1, z, X, Y, Z, sX, sY, sZ, dn); g += dn[1] / fmaxf(m, delta); }
                if (z > 0) { const float m = tv_diffs(v, x, y, z - 1, X, Y, Z, sX, sY, sZ, dn); g += dn[2] / fmaxf(m, delta); }
            }
        }
        grad[idx] = g;
    }
    if (value) {
        __shared__ double red[8];
        r = warp_sum(r);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = r;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < 8; w++) tot += red[w];
            if (tot != 0.0) atomicAdd(value, tot);
        }
    }
}

// Nesterov momentum (reading S22): v <- m v - eta g;  c <- c + v
__global__ void nesterov_kernel(float *__restrict__ c, float *__restrict__ v, const float *__restrict__ g, float eta, float m, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const float vn = fmaf(m, v[i], -eta * g[i]);
        v[i] = vn;
        c[i] += vn;
    }
}

// preconditioned update c <- c - eta * pre (.) g
__global__ void axpy_precond_kernel(float *__restrict__ c, const float *__restrict__ g, const float *__restrict__ pre, float eta, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) c[i] = fmaf(-eta * pre[i], g[i], c[i]);
}

// ================================================================================================
// host-side dispatch
// ================================================================================================
namespace {

mm_status check_launch(const char *what)
{
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        mm_set_error(std::string(what) + ": " + cudaGetErrorString(e));
        return MM_ERR_CUDA;
    }
    g_launches.fetch_add(1);
    return MM_OK;
}

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

mm_status check_common(const mm_geometry *g, int K, int ldk, const char *who)
{
    if (!g) { mm_set_error(std::string(who) + ": NULL geometry"); return MM_ERR_NULL; }
    if (!g->d_table) { mm_set_error(std::string(who) + ": geometry was created without a CUDA device (no CPU fallback)"); return MM_ERR_CUDA; }
    if (K < 1 || ldk < K) { mm_set_error(std::string(who) + ": need 1 <= K <= ldk"); return MM_ERR_SHAPE; }
    if (K > 256 || ldk > 256) { mm_set_error(std::string(who) + ": K, ldk > 256 are not supported"); return MM_ERR_UNSUPPORTED; }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != g->device) {
        cudaGetLastError();
        mm_set_error(std::string(who) + ": the geometry was created on CUDA device " + std::to_string(g->device) +
                     ", the current device is " + std::to_string(dev));
        return MM_ERR_VALUE;
    }
    return MM_OK;
}

template <int VEC, int G, int NQ, int DMAX, int MODE>
void launch_fwd(const FwdArgs &a, cudaStream_t st)
{
    constexpr int RPB = 256 / G;
    constexpr int TK = (RPB >= 64) ? 8 : (RPB >= 32 ? FWD_TK : (RPB >= 4 ? 4 : RPB));
    constexpr int TJ = RPB / TK;
    const long long tiles = (long long)a.P * ((a.J + TJ - 1) / TJ) * ((a.Kd + TK - 1) / TK);
    if constexpr ((VEC == 4 && G >= FWD_U) || (VEC == 8 && G >= 4)) {
        // cooperative march: tap offsets are 32-bit lane-vector indices
        if ((long long)a.X * a.Y * a.Z * (a.ldk / VEC) < (1LL << 31)) {
            john_forward_kernel<VEC, G, NQ, DMAX, MODE, true><<<(unsigned)tiles, 256, 0, st>>>(a);
            return;
        }
    }
    john_forward_kernel<VEC, G, NQ, DMAX, MODE, false><<<(unsigned)tiles, 256, 0, st>>>(a);
}

// ldk = 48 (K = 45, configs 3 and 5): march a copy of the volume with an all-zero record appended (stream-ordered
// scratch from the library's pool; the copy costs 2 x 3.2 GB of traffic on config 5, ~1 ms before a 175 ms march) in
// the nested-difference form (LERP).  Returns false if the scratch could not be had; the caller then takes the
// weighted-FMA path on the caller's own buffer.
template <int DMAX, int MODE>
bool launch_fwd_lerp(const FwdArgs &a, cudaStream_t st)
{
    const long long nvox = (long long)a.X * a.Y * a.Z;
    if ((nvox + 1) * 12 >= (1LL << 31)) return false;           // tap offsets are 32-bit float4 indices
    float *scratch = nullptr;
    if (mm_scratch_alloc((void **)&scratch, (size_t)(nvox + 1) * 48 * sizeof(float), st) != cudaSuccess) { cudaGetLastError(); return false; }
    bool ok = cudaMemcpyAsync(scratch, a.vol, (size_t)nvox * 48 * sizeof(float), cudaMemcpyDeviceToDevice, st) == cudaSuccess &&
              cudaMemsetAsync(scratch + nvox * 48, 0, 48 * sizeof(float), st) == cudaSuccess;
    if (ok) {
        FwdArgs b = a;
        b.vol = scratch; b.zero_vox = (int)nvox;
        constexpr int TK = 8, TJ = 8;                           // 64 rays per block (G = 4)
        const long long tiles = (long long)a.P * ((a.J + TJ - 1) / TJ) * ((a.Kd + TK - 1) / TK);
        john_forward_kernel<4, 4, 3, DMAX, MODE, true, true><<<(unsigned)tiles, 256, 0, st>>>(b);
    } else {
        cudaGetLastError();
    }
    mm_scratch_free(scratch, st);
    return ok;
}

template <int DMAX, int MODE>
mm_status dispatch_fwd(const FwdArgs &a, bool vec, cudaStream_t st)
{
    static const bool lerp_off = getenv("MM_DISABLE_LERP") != nullptr;     // debugging switch: weighted FMAs on the caller's buffer
    if (vec && a.ldk == 48 && !lerp_off && launch_fwd_lerp<DMAX, MODE>(a, st))
        return check_launch("john_forward_kernel (nested-difference form)");
    // 48 floats per voxel (K = 45, configs 3 and 5) = 12 float4 = 4 lanes x 3: every lane's load is used.  The
    // 8 x 32-byte layout below would idle 2 lanes in 8, and the register write-back of a load costs the same
    // 8 wavefronts whether or not its lanes carry new data (profiles/r01_ncu_c5_v5.md): 198 -> 191 ms on config 5.
    if (vec && a.ldk == 48 && (!FWD_MIX48 || (reinterpret_cast<uintptr_t>(a.vol) & 31u) == 0)) { launch_fwd<4, 4, 3, DMAX, MODE>(a, st); return check_launch("john_forward_kernel"); }
    // 32-byte lanes (LDG.E.256): 4 lanes cover up to 32 channels, 8 lanes up to 64, 16 lanes up to 128
    if (vec && a.ldk % 8 == 0 && a.ldk >= 24 && a.ldk <= 128 && (reinterpret_cast<uintptr_t>(a.vol) & 31u) == 0 &&
        (reinterpret_cast<uintptr_t>(a.proj) & 31u) == 0) {
        if (a.ldk <= 32) launch_fwd<8, 4, 1, DMAX, MODE>(a, st);
        else if (a.ldk <= 64) launch_fwd<8, 8, 1, DMAX, MODE>(a, st);
        else launch_fwd<8, 16, 1, DMAX, MODE>(a, st);
        return check_launch("john_forward_kernel");
    }
    if (vec) {
        const int lpv = a.ldk / 4;
        if (lpv <= 1) launch_fwd<4, 1, 1, DMAX, MODE>(a, st);
        else if (lpv <= 2) launch_fwd<4, 2, 1, DMAX, MODE>(a, st);
        else if (lpv <= 4) launch_fwd<4, 4, 1, DMAX, MODE>(a, st);
        else if (lpv <= 8) launch_fwd<4, 8, 1, DMAX, MODE>(a, st);
        else if (lpv <= 16) launch_fwd<4, 16, 1, DMAX, MODE>(a, st);
        else if (lpv <= 32) launch_fwd<4, 32, 1, DMAX, MODE>(a, st);
        else launch_fwd<4, 32, 2, DMAX, MODE>(a, st);
    } else {
        if (a.ldk <= 32) launch_fwd<1, 32, 1, DMAX, MODE>(a, st);
        else launch_fwd<1, 32, 8, DMAX, MODE>(a, st);
    }
    return check_launch("john_forward_kernel");
}

template <int MODE>
mm_status dispatch_fwd_d(const FwdArgs &a, bool vec, cudaStream_t st)
{
    if constexpr (MODE == 0) return dispatch_fwd<1, MODE>(a, vec, st);
    else if (a.D <= 8) return dispatch_fwd<8, MODE>(a, vec, st);
    if (a.D <= 16) return dispatch_fwd<16, MODE>(a, vec, st);
    return dispatch_fwd<32, MODE>(a, vec, st);
}

void fill_fwd(FwdArgs &a, const mm_geometry *g, const float *vol, int K, int ldk)
{
    a.tab = g->d_table; a.vol = vol; a.zero_vox = 0; a.K = K; a.ldk = ldk;
    a.X = g->shape[0]; a.Y = g->shape[1]; a.Z = g->shape[2]; a.J = g->J; a.Kd = g->Kd; a.P = g->P;
    a.proj = nullptr; a.B = nullptr; a.D = 0; a.data = nullptr; a.weights = nullptr; a.sino = nullptr; a.loss = nullptr;
    a.huber = 0.f;
}

void fill_adj(AdjArgs &a, const mm_geometry *g, const float *src, const float *B, float *out, int K, int ldk, int D)
{
    a.tab = g->d_table; a.src = src; a.B = B; a.out = out; a.K = K; a.ldk = ldk; a.D = D;
    a.X = g->shape[0]; a.Y = g->shape[1]; a.Z = g->shape[2]; a.J = g->J; a.Kd = g->Kd; a.P = g->P;
    a.vec_ok = 0; a.bilinear = 0;
    a.vox_begin = 0; a.vox_end = (long long)a.X * a.Y * a.Z;
}

template <int VEC, int G, int NQ>
void launch_adj(const AdjArgs &a, cudaStream_t st)
{
    constexpr int VPB = 256 / G;
    const long long nvox = (long long)a.X * a.Y * a.Z;
    john_adjoint_kernel<VEC, G, NQ><<<(unsigned)((nvox + VPB - 1) / VPB), 256, 0, st>>>(a);
}

template <int KMAX>
mm_status launch_adj_fused(const AdjArgs &a, cudaStream_t st)
{
    const long long nvox = a.vox_end - a.vox_begin;
    if (nvox <= 0) return MM_OK;
    dim3 grid((unsigned)((nvox + 127) / 128), (unsigned)((a.ldk + KMAX - 1) / KMAX));
    // chunks past K only need to zero the pad channels; they still run the (cheap for them) common path
    if (a.D <= 8) adjoint_fused_kernel<KMAX, 8><<<grid, 128, 0, st>>>(a);
    else if (a.D <= 16) adjoint_fused_kernel<KMAX, 16><<<grid, 128, 0, st>>>(a);
    else if constexpr (KMAX <= 32) adjoint_fused_kernel<KMAX, 32><<<grid, 128, 0, st>>>(a);
    else { mm_set_error("adjoint_fused_kernel: no instantiation"); return MM_ERR_UNSUPPORTED; }
    return check_launch("adjoint_fused_kernel");
}

// vox_end < 0: the whole volume; otherwise only voxels [vox_begin, vox_end) of `out` are written
mm_status run_adjoint_fused(const mm_geometry *g, const float *B, const float *sino, int K, int ldk, int D,
                            float *out, cudaStream_t st, int bilinear = 0, long long vox_begin = 0, long long vox_end = -1)
{
    AdjArgs a;
    fill_adj(a, g, sino, B, out, K, ldk, D);
    a.bilinear = bilinear;
    if (vox_end >= 0) { a.vox_begin = vox_begin; a.vox_end = vox_end; }
    a.vec_ok = (D % 4 == 0) && aligned16(sino);
    static const bool tc_off = getenv("MM_DISABLE_TC") != nullptr;     // debugging switch: CUDA-core contraction
    static const bool brick_off = getenv("MM_DISABLE_BRICK") != nullptr;   // debugging switch: round-1 global-load gather
    if (!tc_off && !brick_off && mm_adjoint_brick_supported(g, a)) {   // primary path: bricks + TMA tiles + tcgen05
        const cudaError_t e = (cudaError_t)mm_adjoint_brick_launch(g, a, st);
        if (e != cudaSuccess) {
            mm_set_error(std::string("adjoint_brick_kernel: ") + cudaGetErrorString(e));
            cudaGetLastError();
            return MM_ERR_CUDA;
        }
        g_launches.fetch_add(2);                                      // bop_prep_kernel + adjoint_brick_kernel
        return MM_OK;
    }
    if (!tc_off && mm_adjoint_tc_supported(a)) {
        const cudaError_t e = (cudaError_t)mm_adjoint_tc_launch(a, st);
        if (e != cudaSuccess) {
            mm_set_error(std::string("adjoint_tc_kernel: ") + cudaGetErrorString(e));
            return MM_ERR_CUDA;
        }
        g_launches.fetch_add(1);
        return MM_OK;
    }
    if (ldk <= 8) return launch_adj_fused<8>(a, st);
    if (ldk <= 16) return launch_adj_fused<16>(a, st);
    if (ldk <= 32) return launch_adj_fused<32>(a, st);
    if (D <= 16) return launch_adj_fused<48>(a, st);
    return launch_adj_fused<32>(a, st);
}

}  // namespace

extern "C" mm_status mm_john_forward(const mm_geometry *g, const float *vol, int32_t K, int32_t ldk, float *proj, void *stream)
{
    mm_status st = check_common(g, K, ldk, "mm_john_forward");
    if (st != MM_OK) return st;
    if (!vol || !proj) { mm_set_error("mm_john_forward: NULL buffer"); return MM_ERR_NULL; }
    FwdArgs a;
    fill_fwd(a, g, vol, K, ldk);
    a.proj = proj;
    const bool vec = (ldk % 4 == 0) && aligned16(vol) && aligned16(proj);
    return dispatch_fwd_d<0>(a, vec, (cudaStream_t)stream);
}

extern "C" mm_status mm_forward(const mm_geometry *g, const float *B, const float *vol, int32_t K, int32_t ldk, int32_t D,
                                float *sino, void *stream)
{
    mm_status st = check_common(g, K, ldk, "mm_forward");
    if (st != MM_OK) return st;
    if (!B || !vol || !sino) { mm_set_error("mm_forward: NULL buffer"); return MM_ERR_NULL; }
    if (D < 1 || D > MM_MAX_D) { mm_set_error("mm_forward: need 1 <= D <= MM_MAX_D"); return MM_ERR_SHAPE; }
    FwdArgs a;
    fill_fwd(a, g, vol, K, ldk);
    a.B = B; a.D = D; a.sino = sino;
    const bool vec = (ldk % 4 == 0) && aligned16(vol);
    return dispatch_fwd_d<1>(a, vec, (cudaStream_t)stream);
}

static mm_status run_john_adjoint(const mm_geometry *g, const float *proj, int32_t K, int32_t ldk, float *vol_out, void *stream,
                                  int bilinear, const char *who)
{
    mm_status st = check_common(g, K, ldk, who);
    if (st != MM_OK) return st;
    if (!proj || !vol_out) { mm_set_error(std::string(who) + ": NULL buffer"); return MM_ERR_NULL; }
    AdjArgs a;
    fill_adj(a, g, proj, nullptr, vol_out, K, ldk, 0);
    a.bilinear = bilinear;
    cudaStream_t cs = (cudaStream_t)stream;
    if ((ldk % 4 == 0) && aligned16(proj) && aligned16(vol_out)) {
        const int lpv = ldk / 4;
        if (lpv <= 1) launch_adj<4, 1, 1>(a, cs);
        else if (lpv <= 2) launch_adj<4, 2, 1>(a, cs);
        else if (lpv <= 4) launch_adj<4, 4, 1>(a, cs);
        else if (lpv <= 8) launch_adj<4, 8, 1>(a, cs);
        else if (lpv <= 16) launch_adj<4, 16, 1>(a, cs);
        else if (lpv <= 32) launch_adj<4, 32, 1>(a, cs);
        else launch_adj<4, 32, 2>(a, cs);
    } else {
        if (ldk <= 32) launch_adj<1, 32, 1>(a, cs);
        else launch_adj<1, 32, 8>(a, cs);
    }
    return check_launch("john_adjoint_kernel");
}

extern "C" mm_status mm_john_adjoint(const mm_geometry *g, const float *proj, int32_t K, int32_t ldk, float *vol_out, void *stream)
{
    return run_john_adjoint(g, proj, K, ldk, vol_out, stream, 0, "mm_john_adjoint");
}

extern "C" mm_status mm_john_backproject(const mm_geometry *g, const float *proj, int32_t K, int32_t ldk, float *vol_out, void *stream)
{
    return run_john_adjoint(g, proj, K, ldk, vol_out, stream, 1, "mm_john_backproject");
}

extern "C" mm_status mm_backproject(const mm_geometry *g, const float *B, const float *sino, int32_t K, int32_t ldk, int32_t D,
                                    float *vol_out, void *stream)
{
    mm_status st = check_common(g, K, ldk, "mm_backproject");
    if (st != MM_OK) return st;
    if (!B || !sino || !vol_out) { mm_set_error("mm_backproject: NULL buffer"); return MM_ERR_NULL; }
    if (D < 1 || D > MM_MAX_D) { mm_set_error("mm_backproject: need 1 <= D <= MM_MAX_D"); return MM_ERR_SHAPE; }
    return run_adjoint_fused(g, B, sino, K, ldk, D, vol_out, (cudaStream_t)stream, 1);
}

extern "C" mm_status mm_adjoint(const mm_geometry *g, const float *B, const float *sino, int32_t K, int32_t ldk, int32_t D,
                                float *vol_out, void *stream)
{
    mm_status st = check_common(g, K, ldk, "mm_adjoint");
    if (st != MM_OK) return st;
    if (!B || !sino || !vol_out) { mm_set_error("mm_adjoint: NULL buffer"); return MM_ERR_NULL; }
    if (D < 1 || D > MM_MAX_D) { mm_set_error("mm_adjoint: need 1 <= D <= MM_MAX_D"); return MM_ERR_SHAPE; }
    return run_adjoint_fused(g, B, sino, K, ldk, D, vol_out, (cudaStream_t)stream);
}

extern "C" mm_status mm_basis_forward(const mm_geometry *g, const float *B, const float *proj, int32_t K, int32_t ldk,
                                      int32_t D, float *sino, void *stream)
{
    mm_status st = check_common(g, K, ldk, "mm_basis_forward");
    if (st != MM_OK) return st;
    if (!B || !proj || !sino) { mm_set_error("mm_basis_forward: NULL buffer"); return MM_ERR_NULL; }
    if (D < 1) { mm_set_error("mm_basis_forward: D < 1"); return MM_ERR_SHAPE; }
    const long long npp = (long long)g->J * g->Kd, total = npp * g->P * D;
    basis_forward_kernel<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)stream>>>(B, proj, sino, K, ldk, D, npp, total);
    return check_launch("basis_forward_kernel");
}

extern "C" mm_status mm_basis_adjoint(const mm_geometry *g, const float *B, const float *sino, int32_t K, int32_t ldk,
                                      int32_t D, float *proj, void *stream)
{
    mm_status st = check_common(g, K, ldk, "mm_basis_adjoint");
    if (st != MM_OK) return st;
    if (!B || !proj || !sino) { mm_set_error("mm_basis_adjoint: NULL buffer"); return MM_ERR_NULL; }
    if (D < 1) { mm_set_error("mm_basis_adjoint: D < 1"); return MM_ERR_SHAPE; }
    const long long npp = (long long)g->J * g->Kd, total = npp * g->P * ldk;
    basis_adjoint_kernel<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)stream>>>(B, sino, proj, K, ldk, D, npp, total);
    return check_launch("basis_adjoint_kernel");
}

static mm_status run_residual_loss(const mm_geometry *g, const float *B, const float *vol, int32_t K, int32_t ldk, int32_t D,
                                   const float *data, const float *weights, float *wr, double *loss, cudaStream_t cs,
                                   const char *who, float huber = 0.f)
{
    mm_status st = check_common(g, K, ldk, who);
    if (st != MM_OK) return st;
    if (!B || !vol || !data || !loss || !wr) { mm_set_error(std::string(who) + ": NULL buffer"); return MM_ERR_NULL; }
    if (D < 1 || D > MM_MAX_D) { mm_set_error(std::string(who) + ": need 1 <= D <= MM_MAX_D"); return MM_ERR_SHAPE; }
    if (cudaMemsetAsync(loss, 0, sizeof(double), cs) != cudaSuccess) {
        mm_set_error(std::string("cudaMemsetAsync(loss): ") + cudaGetErrorString(cudaGetLastError()));
        return MM_ERR_CUDA;
    }
    FwdArgs a;
    fill_fwd(a, g, vol, K, ldk);
    a.B = B; a.D = D; a.data = data; a.weights = weights; a.sino = wr; a.loss = loss; a.huber = huber;
    const bool vec = (ldk % 4 == 0) && aligned16(vol);
    return dispatch_fwd_d<2>(a, vec, cs);                     // a3 + a4 + a5
}

extern "C" mm_status mm_residual_loss(const mm_geometry *g, const float *B, const float *vol, int32_t K, int32_t ldk, int32_t D,
                                      const float *data, const float *weights, float *wr, double *loss, void *stream)
{
    return run_residual_loss(g, B, vol, K, ldk, D, data, weights, wr, loss, (cudaStream_t)stream, "mm_residual_loss");
}

extern "C" mm_status mm_loss_gradient(const mm_geometry *g, const float *B, const float *vol, int32_t K, int32_t ldk, int32_t D,
                                      const float *data, const float *weights, float *grad, double *loss,
                                      float *wr_workspace, void *stream)
{
    if (!grad) { mm_set_error("mm_loss_gradient: NULL buffer"); return MM_ERR_NULL; }
    cudaStream_t cs = (cudaStream_t)stream;
    mm_status st = run_residual_loss(g, B, vol, K, ldk, D, data, weights, wr_workspace, loss, cs, "mm_loss_gradient");   // phase 1
    if (st != MM_OK) return st;
    if (g_phase_event && cudaEventRecord(g_phase_event, cs) != cudaSuccess) {
        mm_set_error(std::string("cudaEventRecord(phase event): ") + cudaGetErrorString(cudaGetLastError()));
        return MM_ERR_CUDA;
    }
    return run_adjoint_fused(g, B, wr_workspace, K, ldk, D, grad, cs);   // phase 2: a6 + a7
}

extern "C" mm_status mm_loss_gradient_huber(const mm_geometry *g, const float *B, const float *vol, int32_t K, int32_t ldk, int32_t D,
                                            const float *data, const float *weights, float delta, float *grad, double *loss,
                                            float *wr_workspace, void *stream)
{
    if (!grad) { mm_set_error("mm_loss_gradient_huber: NULL buffer"); return MM_ERR_NULL; }
    if (!(delta > 0.f)) { mm_set_error("mm_loss_gradient_huber: delta must be positive"); return MM_ERR_VALUE; }
    cudaStream_t cs = (cudaStream_t)stream;
    mm_status st = run_residual_loss(g, B, vol, K, ldk, D, data, weights, wr_workspace, loss, cs, "mm_loss_gradient_huber", delta);
    if (st != MM_OK) return st;
    return run_adjoint_fused(g, B, wr_workspace, K, ldk, D, grad, cs);
}

extern "C" mm_status mm_reciprocal(float *x, int64_t n, float floor_, void *stream)
{
    if (!x) { mm_set_error("mm_reciprocal: NULL buffer"); return MM_ERR_NULL; }
    if (n < 0) { mm_set_error("mm_reciprocal: n < 0"); return MM_ERR_SHAPE; }
    if (n == 0) return MM_OK;
    reciprocal_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(x, floor_, (long long)n);
    return check_launch("reciprocal_kernel");
}

extern "C" mm_status mm_laplacian(const mm_geometry *g, const float *vol, int32_t K, int32_t ldk, float *vol_out, void *stream)
{
    mm_status st = check_common(g, K, ldk, "mm_laplacian");
    if (st != MM_OK) return st;
    if (!vol || !vol_out) { mm_set_error("mm_laplacian: NULL buffer"); return MM_ERR_NULL; }
    if (vol == vol_out) { mm_set_error("mm_laplacian: in and out must differ"); return MM_ERR_VALUE; }
    const int X = g->shape[0], Y = g->shape[1], Z = g->shape[2];
    const bool vec = (ldk % 4 == 0) && aligned16(vol) && aligned16(vol_out);
    const long long total = (long long)X * Y * Z * (vec ? ldk / 4 : ldk);
    const unsigned blocks = (unsigned)((total + 255) / 256);
    if (vec) laplacian_kernel<4><<<blocks, 256, 0, (cudaStream_t)stream>>>(vol, vol_out, X, Y, Z, ldk, K);
    else laplacian_kernel<1><<<blocks, 256, 0, (cudaStream_t)stream>>>(vol, vol_out, X, Y, Z, ldk, K);
    return check_launch("laplacian_kernel");
}

extern "C" mm_status mm_derived_quantities(const mm_geometry *g, const float *vol, int32_t K, int32_t ldk, float *mean, float *moments,
                                           float *eigenvalues, float *eigenvectors, float *fa, void *stream)
{
    mm_status st = check_common(g, K, ldk, "mm_derived_quantities");
    if (st != MM_OK) return st;
    if (!vol) { mm_set_error("mm_derived_quantities: NULL volume"); return MM_ERR_NULL; }
    const long long nvox = (long long)g->shape[0] * g->shape[1] * g->shape[2];
    derived_kernel<<<(unsigned)((nvox + 127) / 128), 128, 0, (cudaStream_t)stream>>>(vol, ldk, K, nvox, mean, moments, eigenvalues,
                                                                                      eigenvectors, fa);
    return check_launch("derived_kernel");
}

extern "C" mm_status mm_regulariser(const mm_geometry *g, int32_t kind, const float *vol, int32_t K, int32_t ldk, float delta,
                                    float *grad_out, double *value, void *stream)
{
    mm_status st = check_common(g, K, ldk, "mm_regulariser");
    if (st != MM_OK) return st;
    if (!vol || !grad_out) { mm_set_error("mm_regulariser: NULL buffer"); return MM_ERR_NULL; }
    if (vol == grad_out) { mm_set_error("mm_regulariser: in and out must differ"); return MM_ERR_VALUE; }
    if (kind != MM_REG_L1 && kind != MM_REG_HUBER && kind != MM_REG_TV) { mm_set_error("mm_regulariser: unknown kind"); return MM_ERR_VALUE; }
    if (kind != MM_REG_L1 && !(delta > 0.f)) { mm_set_error("mm_regulariser: delta must be positive"); return MM_ERR_VALUE; }
    cudaStream_t cs = (cudaStream_t)stream;
    if (value && cudaMemsetAsync(value, 0, sizeof(double), cs) != cudaSuccess) {
        mm_set_error(std::string("cudaMemsetAsync(value): ") + cudaGetErrorString(cudaGetLastError()));
        return MM_ERR_CUDA;
    }
    const int X = g->shape[0], Y = g->shape[1], Z = g->shape[2];
    const long long total = (long long)X * Y * Z * ldk;
    regulariser_kernel<<<(unsigned)((total + 255) / 256), 256, 0, cs>>>(vol, grad_out, value, kind, delta, X, Y, Z, ldk, K);
    return check_launch("regulariser_kernel");
}

extern "C" mm_status mm_nesterov_step(float *c, float *v, const float *grad, float eta, float momentum, int64_t n, void *stream)
{
    if (!c || !v || !grad) { mm_set_error("mm_nesterov_step: NULL buffer"); return MM_ERR_NULL; }
    if (n < 0) { mm_set_error("mm_nesterov_step: n < 0"); return MM_ERR_SHAPE; }
    if (n == 0) return MM_OK;
    nesterov_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(c, v, grad, eta, momentum, (long long)n);
    return check_launch("nesterov_kernel");
}

extern "C" mm_status mm_axpy_precond(float *c, const float *grad, const float *pre, float eta, int64_t n, void *stream)
{
    if (!c || !grad || !pre) { mm_set_error("mm_axpy_precond: NULL buffer"); return MM_ERR_NULL; }
    if (n < 0) { mm_set_error("mm_axpy_precond: n < 0"); return MM_ERR_SHAPE; }
    if (n == 0) return MM_OK;
    axpy_precond_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(c, grad, pre, eta, (long long)n);
    return check_launch("axpy_precond_kernel");
}

extern "C" mm_status mm_axpy(float *c, const float *grad, float eta, int64_t n, void *stream)
{
    if (!c || !grad) { mm_set_error("mm_axpy: NULL buffer"); return MM_ERR_NULL; }
    if (n < 0) { mm_set_error("mm_axpy: n < 0"); return MM_ERR_SHAPE; }
    if (n == 0) return MM_OK;
    axpy_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(c, grad, eta, (long long)n);
    return check_launch("axpy_kernel");
}

// Device workspace of the host-buffer call: one grow-only arena and one stream per process, kept between calls
// (cudaMalloc/cudaFree of 7 GB cost 20-330 ms per call on config 5, more than the copies); mm_host_workspace_release
// frees it.  Calls are serialised by the mutex.
namespace {
struct HostWorkspace {
    std::mutex mu;
    char *base = nullptr;
    size_t bytes = 0;
    cudaStream_t stream = nullptr, copy_stream = nullptr;
    cudaEvent_t range_done = nullptr;
    int device = -1;
} g_hws;

void hws_free_locked()
{
    if (g_hws.base) cudaFree(g_hws.base);
    if (g_hws.stream) cudaStreamDestroy(g_hws.stream);
    if (g_hws.copy_stream) cudaStreamDestroy(g_hws.copy_stream);
    if (g_hws.range_done) cudaEventDestroy(g_hws.range_done);
    g_hws.base = nullptr; g_hws.bytes = 0; g_hws.stream = g_hws.copy_stream = nullptr; g_hws.range_done = nullptr; g_hws.device = -1;
}
}   // namespace

extern "C" mm_status mm_host_workspace_release(void)
{
    std::lock_guard<std::mutex> lock(g_hws.mu);
    hws_free_locked();
    return MM_OK;
}

extern "C" mm_status mm_workspace_release(void)
{
    {
        std::lock_guard<std::mutex> lock(g_hws.mu);
        hws_free_locked();
    }
    mm_scratch_trim();
    return MM_OK;
}

extern "C" mm_status mm_loss_gradient_host(const mm_geometry *g, const float *h_B, const float *h_vol, int32_t K, int32_t ldk,
                                           int32_t D, const float *h_data, const float *h_weights, float *h_grad, double *h_loss)
{
    mm_status st = check_common(g, K, ldk, "mm_loss_gradient_host");
    if (st != MM_OK) return st;
    if (!h_B || !h_vol || !h_data || !h_grad || !h_loss) { mm_set_error("mm_loss_gradient_host: NULL buffer"); return MM_ERR_NULL; }
    if (D < 1 || D > MM_MAX_D) { mm_set_error("mm_loss_gradient_host: need 1 <= D <= MM_MAX_D"); return MM_ERR_SHAPE; }
    const size_t nvol = (size_t)g->shape[0] * g->shape[1] * g->shape[2] * ldk * sizeof(float);
    const size_t nsino = (size_t)g->P * g->J * g->Kd * D * sizeof(float);
    const size_t nB = (size_t)g->P * K * D * sizeof(float);
    auto up = [](size_t n) { return (n + 255) & ~(size_t)255; };          // every buffer 256-byte aligned
    const size_t need = 2 * up(nvol) + (h_weights ? 3 : 2) * up(nsino) + up(nB) + 256;
    mm_status rc = MM_OK;
    cudaError_t e = cudaSuccess;
#define MM_TRY(call, code)                                                              \
    if (rc == MM_OK && (e = (call)) != cudaSuccess) {                                    \
        mm_set_error(std::string(#call) + ": " + cudaGetErrorString(e));                \
        cudaGetLastError();                                                             \
        rc = code;                                                                      \
    }
    std::lock_guard<std::mutex> lock(g_hws.mu);
    int dev = -1;
    MM_TRY(cudaGetDevice(&dev), MM_ERR_CUDA);
    if (rc == MM_OK && (dev != g_hws.device || need > g_hws.bytes)) {
        hws_free_locked();
        MM_TRY(cudaMalloc((void **)&g_hws.base, need), MM_ERR_ALLOC);
        MM_TRY(cudaStreamCreate(&g_hws.stream), MM_ERR_CUDA);
        MM_TRY(cudaStreamCreate(&g_hws.copy_stream), MM_ERR_CUDA);
        MM_TRY(cudaEventCreateWithFlags(&g_hws.range_done, cudaEventDisableTiming), MM_ERR_CUDA);
        if (rc == MM_OK) { g_hws.bytes = need; g_hws.device = dev; } else hws_free_locked();
    }
    if (rc != MM_OK) return rc;
    char *p = g_hws.base;
    auto take = [&](size_t n) { char *q = p; p += up(n); return q; };
    float *dvol = (float *)take(nvol), *dgrad = (float *)take(nvol), *ddata = (float *)take(nsino), *dwr = (float *)take(nsino);
    float *dw = h_weights ? (float *)take(nsino) : nullptr, *dB = (float *)take(nB);
    double *dloss = (double *)take(sizeof(double));
    cudaStream_t cs = g_hws.stream;
    MM_TRY(cudaMemcpyAsync(dB, h_B, nB, cudaMemcpyHostToDevice, cs), MM_ERR_CUDA);
    MM_TRY(cudaMemcpyAsync(dvol, h_vol, nvol, cudaMemcpyHostToDevice, cs), MM_ERR_CUDA);
    MM_TRY(cudaMemcpyAsync(ddata, h_data, nsino, cudaMemcpyHostToDevice, cs), MM_ERR_CUDA);
    if (h_weights) MM_TRY(cudaMemcpyAsync(dw, h_weights, nsino, cudaMemcpyHostToDevice, cs), MM_ERR_CUDA);
    if (rc == MM_OK) rc = run_residual_loss(g, dB, dvol, K, ldk, D, ddata, dw, dwr, dloss, cs, "mm_loss_gradient_host");   // phase 1
    MM_TRY(cudaMemcpyAsync(h_loss, dloss, sizeof(double), cudaMemcpyDeviceToHost, cs), MM_ERR_CUDA);
    // phase 2 in ranges of voxels: the device->host copy of a finished range runs on the copy stream under the
    // next range's kernel (the 3.2 GB gradient of config 5 takes ~60 ms to copy, the kernel 123 ms)
    const long long nvox = (long long)g->shape[0] * g->shape[1] * g->shape[2];
    const long long plane = (long long)g->shape[1] * g->shape[2];
    const int X = g->shape[0];
    const int nrange = X >= 32 ? 8 : 1;                                   // ranges of whole x-planes, multiples of 4 planes
    cudaStream_t cp = g_hws.copy_stream;
    for (int c = 0; c < nrange && rc == MM_OK; c++) {
        const long long b = (long long)((X * c / nrange) & ~3) * plane;
        const long long e2 = (c + 1 == nrange) ? nvox : (long long)((X * (c + 1) / nrange) & ~3) * plane;
        rc = run_adjoint_fused(g, dB, dwr, K, ldk, D, dgrad, cs, 0, b, e2);
        MM_TRY(cudaEventRecord(g_hws.range_done, cs), MM_ERR_CUDA);
        MM_TRY(cudaStreamWaitEvent(cp, g_hws.range_done, 0), MM_ERR_CUDA);
        MM_TRY(cudaMemcpyAsync(h_grad + b * ldk, dgrad + b * ldk, (size_t)(e2 - b) * ldk * sizeof(float), cudaMemcpyDeviceToHost, cp),
               MM_ERR_CUDA);
    }
    if (rc == MM_OK) { MM_TRY(cudaStreamSynchronize(cs), MM_ERR_CUDA); } else cudaStreamSynchronize(cs);
    if (rc == MM_OK) { MM_TRY(cudaStreamSynchronize(cp), MM_ERR_CUDA); } else cudaStreamSynchronize(cp);
#undef MM_TRY
    return rc;
}
