// mm_sparse.cu — NEXT-2: the forward model with a SPARSE reciprocal-space map ("a modified version of the
// John transform that calculates the reciprocal-space and real-space projection operations simultaneously within one
// kernel, using a sparse approximation to the reciprocal-space mapping"; reading S26 for what the approximation is).
//
// Where sparsity pays on this hardware.  The dense fused forward marches ALL K channels of every tap and is bound by
// the bytes that cross the L1 data pipe into registers.  With a nearest-neighbour basis
// or a thresholded one only a few channels i have a non-zero row B[s][i][:] for a given projection s (K = 162
// directions, D = 8 segments, 8 quadrature points: ~20 of 162).  The sparse kernel marches only those: one warp per
// ray, lane l owns active channel idx[s][l], four scalar taps per slab — one 128-byte register write-back per tap
// instead of five.  The K x D contraction of the adjoint stays dense on the tensor cores (a zero row costs nothing
// there: 3 x 162 x 8 MACs per voxel-projection are ~2 ms of tensor time on the 100^3 / 240-projection case).
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#include <algorithm>
#include <new>
#include <string>
#include <vector>

#include "mm_internal.h"

struct mm_sparse_plan {
    int P, K, D;
    int max_active;                 // largest number of active channels of a projection
    double mean_active;
    std::vector<int> h_count;       // [P]
    int *d_idx;                     // [P][slots]: active channels of projection s, ascending; unused slots hold 0
    int *d_count;                   // [P]
    int slots;                      // max_active rounded up to a multiple of 32
    int device;
};

namespace {

#define SP_FX_BITS 40
#define SP_FX_ONE 1099511627776.0
#define SP_FX_INV 2.3283064365386963e-10f

struct SparseArgs {
    const MMProj *tab;
    const float *vol;
    const int *idx, *count;
    int slots;
    int K, ldk, X, Y, Z, J, Kd, P, D;
    const float *B, *data, *weights;
    float *sino;                    // MODE 1: model sinogram; MODE 2: wr
    double *loss;
};

__device__ __forceinline__ void sp_clip(double A, double s, int N, double &lo, double &hi)
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

// One warp per ray; lane l marches channels idx[l], idx[l + 32], ... (NQ of them).  Same Joseph arithmetic as the dense
// kernels (24.40 fixed-point positions, fp32 rounds of 4 slabs flushed into fp64 totals, fp64 epilogue); tap offsets
// are 32-bit float indices (the host refuses larger volumes).
template <int NQ, int DMAX, int MODE>
__global__ void __launch_bounds__(256) john_forward_sparse_kernel(const SparseArgs a)
{
    constexpr int TK = 4, TJ = 2;                                  // 8 rays (warps) per block
    const int lane = threadIdx.x & 31, r = threadIdx.x >> 5;
    const int tiles_k = (a.Kd + TK - 1) / TK, tiles_j = (a.J + TJ - 1) / TJ;
    const int tpp = tiles_k * tiles_j;
    const int s = blockIdx.x / tpp;
    int tile = blockIdx.x - s * tpp;
    const int tk = tile % tiles_k, tj = tile / tiles_k;
    const int j = tj * TJ + r / TK, k = tk * TK + r % TK;
    const bool ray_ok = (j < a.J) && (k < a.Kd);
    const MMProj *pg = a.tab + s;
    const int m = pg->m, u = pg->u, v = pg->v;
    const int Nm = (m == 0) ? a.X : (m == 1 ? a.Y : a.Z);
    const int Nu = (u == 0) ? a.X : a.Y, Nv = (v == 2) ? a.Z : a.Y;
    const long long sX = (long long)a.Y * a.Z * a.ldk, sY = (long long)a.Z * a.ldk, sZ = a.ldk;
    const long long sM = (m == 0) ? sX : (m == 1 ? sY : sZ);
    const long long sU = (u == 0) ? sX : sY, sV = (v == 2) ? sZ : sY;
    const int na = a.count[s];
    int ch[NQ];
    bool on[NQ];
#pragma unroll
    for (int t = 0; t < NQ; t++) {
        on[t] = lane + 32 * t < na;
        ch[t] = on[t] ? a.idx[(long long)s * a.slots + lane + 32 * t] : 0;
    }
    float acc[NQ];
    double tot[NQ];
#pragma unroll
    for (int t = 0; t < NQ; t++) { acc[t] = 0.f; tot[t] = 0.0; }
    // Cooperative march (as in the dense kernel): the 32 lanes work out the taps of 32 consecutive slabs, one slab
    // each, park them in shared memory, and the warp then streams through the round doing only loads and FMAs.
    __shared__ int4 tap_o[8][33];
    __shared__ float4 tap_w[8][33];
    int n0 = 0, n1 = -1;
    long long pu0 = 0, pv0 = 0;
    if (ray_ok) {
        const double Au = pg->Cu + (double)j * pg->Mju + (double)k * pg->Mku;
        const double Av = pg->Cv + (double)j * pg->Mjv + (double)k * pg->Mkv;
        double lo = 0.0, hi = (double)(Nm - 1);
        sp_clip(Au, pg->su, Nu, lo, hi);
        sp_clip(Av, pg->sv, Nv, lo, hi);
        n0 = (int)ceil(lo); n1 = (int)floor(hi);
        pu0 = (long long)floor(Au * SP_FX_ONE);
        pv0 = (long long)floor(Av * SP_FX_ONE);
    }
    const long long su_fx = pg->su_fx, sv_fx = pg->sv_fx;
    for (int nb = n0; nb <= n1; nb += 32) {
        {   // lane l: taps of slab nb + l (offsets in floats from the volume base; taps outside the volume: weight 0, offset 0)
            const int n = nb + lane;
            int4 o = make_int4(0, 0, 0, 0);
            float4 wgt = make_float4(0.f, 0.f, 0.f, 0.f);
            if (n <= n1) {
                const long long pu = pu0 + (long long)n * su_fx, pv = pv0 + (long long)n * sv_fx;
                const int iu = (int)(pu >> SP_FX_BITS), iv = (int)(pv >> SP_FX_BITS);
                const float fu = (float)(unsigned int)(pu >> (SP_FX_BITS - 32)) * SP_FX_INV;
                const float fv = (float)(unsigned int)(pv >> (SP_FX_BITS - 32)) * SP_FX_INV;
                const bool u0 = (unsigned)iu < (unsigned)Nu, u1 = (unsigned)(iu + 1) < (unsigned)Nu;
                const bool v0 = (unsigned)iv < (unsigned)Nv, v1 = (unsigned)(iv + 1) < (unsigned)Nv;
                const int b0 = n * (int)sM + (u0 ? iu * (int)sU : 0), b1 = n * (int)sM + (u1 ? (iu + 1) * (int)sU : 0);
                const int c0 = v0 ? iv * (int)sV : 0, c1 = v1 ? (iv + 1) * (int)sV : 0;
                o = make_int4(b0 + c0, b1 + c0, b0 + c1, b1 + c1);
                wgt = make_float4((u0 && v0) ? (1.f - fu) * (1.f - fv) : 0.f, (u1 && v0) ? fu * (1.f - fv) : 0.f,
                                  (u0 && v1) ? (1.f - fu) * fv : 0.f, (u1 && v1) ? fu * fv : 0.f);
            }
            tap_o[r][lane] = o;
            tap_w[r][lane] = wgt;
        }
        __syncwarp();
        const int cnt = min(32, n1 - nb + 1);
        for (int i = 0; i < cnt; i += 4) {                         // 4 slabs (16 taps per channel) in flight; slabs past n1 carry weight 0
            float c[4][NQ][4];
            float4 w4[4];
#pragma unroll
            for (int uu = 0; uu < 4; uu++) {
                const int4 o = tap_o[r][i + uu];
                w4[uu] = tap_w[r][i + uu];
#pragma unroll
                for (int t = 0; t < NQ; t++) {
                    c[uu][t][0] = on[t] ? __ldg(a.vol + o.x + ch[t]) : 0.f;
                    c[uu][t][1] = on[t] ? __ldg(a.vol + o.y + ch[t]) : 0.f;
                    c[uu][t][2] = on[t] ? __ldg(a.vol + o.z + ch[t]) : 0.f;
                    c[uu][t][3] = on[t] ? __ldg(a.vol + o.w + ch[t]) : 0.f;
                }
            }
#pragma unroll
            for (int uu = 0; uu < 4; uu++)
#pragma unroll
                for (int t = 0; t < NQ; t++) {
                    acc[t] = fmaf(w4[uu].x, c[uu][t][0], acc[t]); acc[t] = fmaf(w4[uu].y, c[uu][t][1], acc[t]);
                    acc[t] = fmaf(w4[uu].z, c[uu][t][2], acc[t]); acc[t] = fmaf(w4[uu].w, c[uu][t][3], acc[t]);
                }
#pragma unroll
            for (int t = 0; t < NQ; t++) { tot[t] += (double)acc[t]; acc[t] = 0.f; }
        }
        __syncwarp();
    }
    // reciprocal-space map restricted to the active rows of B_s (Eq. 6), residual, loss: fp64, reduced over the warp
    const double w = pg->w64;
    double part[DMAX];
#pragma unroll
    for (int c = 0; c < DMAX; c++) part[c] = 0.0;
    const float *Bs = a.B + (long long)s * a.K * a.D;
#pragma unroll
    for (int t = 0; t < NQ; t++) {
        if (on[t]) {
            const double pv_ = w * tot[t];
#pragma unroll
            for (int c = 0; c < DMAX; c++)
                if (c < a.D) part[c] = fma((double)__ldg(Bs + (long long)ch[t] * a.D + c), pv_, part[c]);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int c = 0; c < DMAX; c++) part[c] += __shfl_xor_sync(0xffffffffu, part[c], o);
    double lsum = 0.0;
    const long long ray = ((long long)s * a.J + j) * a.Kd + k;
#pragma unroll
    for (int c = 0; c < DMAX; c++) {
        if ((c & 31) == lane && c < a.D && ray_ok) {
            const long long o = ray * a.D + c;
            if (MODE == 1) {
                a.sino[o] = (float)part[c];
            } else {
                const double res = part[c] - (double)__ldg(a.data + o);
                const double wt = a.weights ? (double)__ldg(a.weights + o) : 1.0;
                a.sino[o] = (float)(wt * res);
                lsum += 0.5 * wt * res * res;
            }
        }
    }
    if (MODE == 2) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) lsum += __shfl_xor_sync(0xffffffffu, lsum, o);
        __shared__ double red[8];
        if (lane == 0) red[r] = lsum;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
#pragma unroll
            for (int i = 0; i < 8; i++) t += red[i];
            if (t != 0.0) atomicAdd(a.loss, t);
        }
    }
}

template <int MODE>
mm_status launch_sparse(const SparseArgs &a, cudaStream_t st, const mm_geometry *g = nullptr, const mm_sparse_plan *p = nullptr)
{
    // first choice: the march on channel-planar copies (mm_sparse_planar.cu); MM_DISABLE_PLANAR keeps the record layout
    static const bool planar_off = getenv("MM_DISABLE_PLANAR") != nullptr;
    if (g && p && !planar_off && mm_sparse_planar_supported(g, a.K, a.ldk, p->max_active)) {
        const cudaError_t e = (cudaError_t)mm_sparse_planar_launch(g, a.idx, a.count, a.slots, p->max_active, a.B, a.vol, a.K, a.ldk, a.D,
                                                                   a.data, a.weights, a.sino, a.loss, MODE, st);
        if (e == cudaSuccess) return MM_OK;
        cudaGetLastError();                                         // e.g. no scratch for the copies: the kernel below needs none
    }
    const long long tiles = (long long)a.P * ((a.J + 1) / 2) * ((a.Kd + 3) / 4);
    const int nq = a.slots / 32;
#define MM_SP_CASE(NQ, DM) john_forward_sparse_kernel<NQ, DM, MODE><<<(unsigned)tiles, 256, 0, st>>>(a)
    if (a.D <= 8) { if (nq <= 1) MM_SP_CASE(1, 8); else if (nq <= 2) MM_SP_CASE(2, 8); else if (nq <= 4) MM_SP_CASE(4, 8); else MM_SP_CASE(8, 8); }
    else if (a.D <= 16) { if (nq <= 1) MM_SP_CASE(1, 16); else if (nq <= 2) MM_SP_CASE(2, 16); else if (nq <= 4) MM_SP_CASE(4, 16); else MM_SP_CASE(8, 16); }
    else { if (nq <= 1) MM_SP_CASE(1, 32); else if (nq <= 2) MM_SP_CASE(2, 32); else if (nq <= 4) MM_SP_CASE(4, 32); else MM_SP_CASE(8, 32); }
#undef MM_SP_CASE
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { mm_set_error(std::string("john_forward_sparse_kernel: ") + cudaGetErrorString(e)); return MM_ERR_CUDA; }
    mm_note_launches(1);
    return MM_OK;
}

mm_status check_sparse(const mm_geometry *g, const mm_sparse_plan *p, int K, int ldk, int D, const char *who)
{
    if (!g || !p) { mm_set_error(std::string(who) + ": NULL geometry or plan"); return MM_ERR_NULL; }
    if (!g->d_table || !p->d_idx) { mm_set_error(std::string(who) + ": no CUDA device (no CPU fallback)"); return MM_ERR_CUDA; }
    if (K != p->K || D != p->D || g->P != p->P) { mm_set_error(std::string(who) + ": K, D or P differ from the plan's"); return MM_ERR_SHAPE; }
    if (ldk < K || D < 1 || D > MM_MAX_D) { mm_set_error(std::string(who) + ": need K <= ldk, 1 <= D <= MM_MAX_D"); return MM_ERR_SHAPE; }
    if ((long long)g->shape[0] * g->shape[1] * g->shape[2] * ldk >= (1LL << 31)) {
        mm_set_error(std::string(who) + ": volumes of 2^31 floats or more are not supported by the sparse path (32-bit tap offsets)");
        return MM_ERR_UNSUPPORTED;
    }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != g->device || dev != p->device) {
        cudaGetLastError();
        mm_set_error(std::string(who) + ": geometry, plan and current device differ");
        return MM_ERR_VALUE;
    }
    return MM_OK;
}

void fill_sparse(SparseArgs &a, const mm_geometry *g, const mm_sparse_plan *p, const float *B, const float *vol, int K, int ldk, int D)
{
    a.tab = g->d_table; a.vol = vol; a.idx = p->d_idx; a.count = p->d_count; a.slots = p->slots;
    a.K = K; a.ldk = ldk; a.X = g->shape[0]; a.Y = g->shape[1]; a.Z = g->shape[2]; a.J = g->J; a.Kd = g->Kd; a.P = g->P; a.D = D;
    a.B = B; a.data = nullptr; a.weights = nullptr; a.sino = nullptr; a.loss = nullptr;
}

}  // namespace

extern "C" mm_status mm_basis_sparsify(const float *h_B, int32_t P, int32_t K, int32_t D, int32_t n_keep, float *h_B_out)
{
    if (!h_B || !h_B_out) { mm_set_error("mm_basis_sparsify: NULL argument"); return MM_ERR_NULL; }
    if (P < 1 || K < 1 || D < 1 || n_keep < 1) { mm_set_error("mm_basis_sparsify: need P, K, D, n_keep >= 1"); return MM_ERR_SHAPE; }
    std::vector<int> order(K);
    for (int s = 0; s < P; s++) {
        const float *Bs = h_B + (size_t)s * K * D;
        float *Os = h_B_out + (size_t)s * K * D;
        for (int c = 0; c < D; c++) {
            for (int i = 0; i < K; i++) order[i] = i;
            // the n_keep largest magnitudes of column c, lowest index first among equals
            std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return fabsf(Bs[(size_t)x * D + c]) > fabsf(Bs[(size_t)y * D + c]); });
            for (int q = 0; q < K; q++) {
                const int i = order[q];
                Os[(size_t)i * D + c] = (q < n_keep) ? Bs[(size_t)i * D + c] : 0.f;
            }
        }
    }
    return MM_OK;
}

extern "C" mm_status mm_sparse_plan_create(const mm_geometry *g, const float *h_B, int32_t K, int32_t D, mm_sparse_plan **out)
{
    if (!g || !h_B || !out) { mm_set_error("mm_sparse_plan_create: NULL argument"); return MM_ERR_NULL; }
    *out = nullptr;
    if (K < 1 || K > 256 || D < 1 || D > MM_MAX_D) { mm_set_error("mm_sparse_plan_create: need 1 <= K <= 256, 1 <= D <= MM_MAX_D"); return MM_ERR_SHAPE; }
    mm_sparse_plan *p = new (std::nothrow) mm_sparse_plan();
    if (!p) { mm_set_error("host allocation failed"); return MM_ERR_ALLOC; }
    p->P = g->P; p->K = K; p->D = D; p->d_idx = nullptr; p->d_count = nullptr; p->device = -1;
    p->h_count.assign(g->P, 0);
    std::vector<std::vector<int>> lists(g->P);
    long long total = 0;
    int mx = 0;
    for (int s = 0; s < g->P; s++) {
        for (int i = 0; i < K; i++) {
            bool any = false;
            for (int c = 0; c < D && !any; c++) any = h_B[((size_t)s * K + i) * D + c] != 0.f;
            if (any) lists[s].push_back(i);
        }
        p->h_count[s] = (int)lists[s].size();
        mx = std::max(mx, p->h_count[s]);
        total += p->h_count[s];
    }
    p->max_active = mx;
    p->mean_active = (double)total / g->P;
    p->slots = std::max(32, (mx + 31) / 32 * 32);
    std::vector<int> flat((size_t)g->P * p->slots, 0);
    for (int s = 0; s < g->P; s++) std::copy(lists[s].begin(), lists[s].end(), flat.begin() + (size_t)s * p->slots);
    if (g->d_table) {                                               // a CUDA device is present
        p->device = g->device;
        cudaError_t e = cudaMalloc((void **)&p->d_idx, flat.size() * sizeof(int));
        if (e == cudaSuccess) e = cudaMalloc((void **)&p->d_count, (size_t)g->P * sizeof(int));
        if (e == cudaSuccess) e = cudaMemcpy(p->d_idx, flat.data(), flat.size() * sizeof(int), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(p->d_count, p->h_count.data(), (size_t)g->P * sizeof(int), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) {
            mm_set_error(std::string("mm_sparse_plan_create: ") + cudaGetErrorString(e));
            cudaGetLastError();
            if (p->d_idx) cudaFree(p->d_idx);
            if (p->d_count) cudaFree(p->d_count);
            delete p;
            return MM_ERR_ALLOC;
        }
    }
    *out = p;
    return MM_OK;
}

extern "C" mm_status mm_sparse_plan_destroy(mm_sparse_plan *p)
{
    if (!p) return MM_OK;
    if (p->d_idx) cudaFree(p->d_idx);
    if (p->d_count) cudaFree(p->d_count);
    delete p;
    return MM_OK;
}

extern "C" mm_status mm_sparse_plan_info(const mm_sparse_plan *p, int32_t *max_active, double *mean_active, int32_t *counts)
{
    if (!p) { mm_set_error("mm_sparse_plan_info: NULL plan"); return MM_ERR_NULL; }
    if (max_active) *max_active = p->max_active;
    if (mean_active) *mean_active = p->mean_active;
    if (counts) std::copy(p->h_count.begin(), p->h_count.end(), counts);
    return MM_OK;
}

extern "C" mm_status mm_forward_sparse(const mm_geometry *g, const mm_sparse_plan *p, const float *B, const float *vol, int32_t K,
                                       int32_t ldk, int32_t D, float *sino, void *stream)
{
    mm_status st = check_sparse(g, p, K, ldk, D, "mm_forward_sparse");
    if (st != MM_OK) return st;
    if (!B || !vol || !sino) { mm_set_error("mm_forward_sparse: NULL buffer"); return MM_ERR_NULL; }
    SparseArgs a;
    fill_sparse(a, g, p, B, vol, K, ldk, D);
    a.sino = sino;
    return launch_sparse<1>(a, (cudaStream_t)stream, g, p);
}

extern "C" mm_status mm_loss_gradient_sparse(const mm_geometry *g, const mm_sparse_plan *p, const float *B, const float *vol, int32_t K,
                                             int32_t ldk, int32_t D, const float *data, const float *weights, float *grad,
                                             double *loss, float *wr_workspace, void *stream)
{
    mm_status st = check_sparse(g, p, K, ldk, D, "mm_loss_gradient_sparse");
    if (st != MM_OK) return st;
    if (!B || !vol || !data || !grad || !loss || !wr_workspace) { mm_set_error("mm_loss_gradient_sparse: NULL buffer"); return MM_ERR_NULL; }
    cudaStream_t cs = (cudaStream_t)stream;
    if (cudaMemsetAsync(loss, 0, sizeof(double), cs) != cudaSuccess) {
        mm_set_error(std::string("cudaMemsetAsync(loss): ") + cudaGetErrorString(cudaGetLastError()));
        return MM_ERR_CUDA;
    }
    SparseArgs a;
    fill_sparse(a, g, p, B, vol, K, ldk, D);
    a.data = data; a.weights = weights; a.sino = wr_workspace; a.loss = loss;
    st = launch_sparse<2>(a, cs, g, p);                             // phase 1: active channels only
    if (st != MM_OK) return st;
    return mm_adjoint(g, B, wr_workspace, K, ldk, D, grad, stream);  // phase 2: dense contraction on the tensor cores
}
