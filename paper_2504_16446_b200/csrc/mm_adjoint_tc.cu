// mm_adjoint_tc.cu — fused adjoint A^T (steps a6 + a7) with the basis contraction on the 5th-gen tensor cores.
//
//   grad[x][i] = sum_s sum_c  ( w_s B[s][i][c] ) * t[x][s][c],      t[x][s][c] = sum_(j,k) Lambda Lambda wr[s][j][k][c]
//
// The gather t (exact transpose of the Joseph forward, reading S9) is irregular and stays on the
// CUDA cores, one thread per voxel.  The contraction over (s,c) is a dense GEMM  [128 voxels x (P*D)] . [(P*D) x ldk]
// (2.17 T FMA on BASELINE config 5, the adjoint's dominant term): each CTA streams its
// 128 x 16 slices of t through shared memory into tcgen05.mma (kind::tf32, M=128, N=ldk, K=8) with the fp32
// accumulators in tensor memory.  Plain TF32 (10-bit mantissa) cannot meet the 1e-5 parity bar, so both operands
// are split x = hi + lo with hi = x truncated to TF32 and lo = x - hi (exact), and three products are issued:
// hi*hi + lo*hi + hi*lo (error ~2^-21 per term).
//
// Shared-memory operand layout (K-major, no swizzle; canonical "interleave" form): a core matrix is 8 rows x 16
// bytes (4 tf32) stored contiguously; element (r, k) of a tile with R rows sits at
//     (k/4) * (R*16) + (r/8) * 128 + (r%8) * 16 + (k%4) * 4          =>  SBO = 128, LBO = R*16
// so thread r writes 16 contiguous bytes per 4 columns and consecutive threads write consecutive 16-byte slots.
#include <cuda_runtime.h>
#include <stdint.h>

#include "mm_internal.h"

namespace {

constexpr int TC_M = 128;          // voxels per CTA = MMA M = TMEM lanes
constexpr int TC_THREADS = 128;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- tensor memory ------------------------------------------------------------------------------------------
template <int COLS>
__device__ __forceinline__ void tmem_alloc(uint32_t *slot_in_smem)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot_in_smem)), "n"(COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
}
template <int COLS>
__device__ __forceinline__ void tmem_dealloc(uint32_t addr)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(addr), "n"(COLS));
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// make generic-proxy shared-memory writes visible to the async proxy (tcgen05.mma reads operands through it)
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- mbarrier -----------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// bounded wait: a lost arrival traps (launch error) instead of hanging the GPU
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    for (uint32_t spin = 0; !mbar_try_wait(bar, parity); spin++)
        if (spin > (1u << 26)) __trap();
}
// all tcgen05.mma issued so far by this thread arrive on `bar` when they have completed
__device__ __forceinline__ void tc_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// ---- descriptors and the MMA --------------------------------------------------------------------------------
// shared-memory matrix descriptor, K-major, no swizzle: start address, LBO (between the two 16-byte K halves),
// SBO (between 8-row groups), all in 16-byte units; bits [46,48) = 1 (sm_100 descriptor version)
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((saddr >> 4) & 0x3fff) | ((uint64_t)((lbo_bytes >> 4) & 0x3fff) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3fff) << 32) | (1ull << 46);
}
// instruction descriptor, kind::tf32: D = F32 (bits 4-5 = 1), A = B = TF32 (bits 7-9, 10-12 = 2), both K-major,
// N/8 at bits 17-22, M/16 at bits 24-28
__host__ __device__ constexpr uint32_t idesc_tf32(int M, int N)
{
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void mma_tf32(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// 32 lanes x 16 consecutive 32-bit columns of tensor memory -> 16 registers per thread (thread = lane)
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16])
{
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; i++) v[i] = __uint_as_float(r[i]);
}

// x = hi + lo with both parts exactly representable in TF32 (1+8+10 bits): hi = x rounded to nearest TF32,
// lo = (x - hi) rounded to nearest TF32.  The tensor core ignores the 13 low mantissa bits of its operands, so
// rounding here (instead of letting it truncate) halves the error and removes its bias: |x - hi - lo| <= 2^-23 |x|.
__device__ __forceinline__ float round_tf32(float x)
{
#ifdef TC_SPLIT_TRUNC
    return __uint_as_float(__float_as_uint(x) & 0xffffe000u);
#else
    return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
#endif
}
__device__ __forceinline__ void split_tf32(float x, float &hi, float &lo)
{
    hi = round_tf32(x);
    lo = round_tf32(x - hi);
}

// the fields of MMProj the voxel gather needs (w_s is folded into the staged B operand)
struct TcProj {
    double Jc, Jx0, Jx1, Jx2, Kc, Kx0, Kx1, Kx2;
    float mju, mku, mjv, mkv, hj, hk;
    int valid, pad;
};

__device__ __forceinline__ void load_proj(TcProj &t, const MMProj *tab, int s, int P)
{
    if (s < P) {
        const MMProj *pg = tab + s;
        t.Jc = pg->Jc; t.Jx0 = pg->Jx[0]; t.Jx1 = pg->Jx[1]; t.Jx2 = pg->Jx[2];
        t.Kc = pg->Kc; t.Kx0 = pg->Kx[0]; t.Kx1 = pg->Kx[1]; t.Kx2 = pg->Kx[2];
        t.mju = pg->mju; t.mku = pg->mku; t.mjv = pg->mjv; t.mkv = pg->mkv;
        t.hj = pg->hj; t.hk = pg->hk;
        t.valid = (pg->hj < 1.5f && pg->hk < 1.5f) ? 2 : 1;      // 2: 3 x 3 window suffices
    } else {
        t.Jc = t.Jx0 = t.Jx1 = t.Jx2 = t.Kc = t.Kx0 = t.Kx1 = t.Kx2 = 0.0;
        t.mju = t.mku = t.mjv = t.mkv = 0.f;
        t.hj = t.hk = -1.f; t.valid = 0;           // empty candidate window
    }
    t.pad = 0;
}

// t[c] = sum over the rays (jj,kk) of projection s that pass within one voxel of (x,y,z) in its slab of
//        Lambda(du) Lambda(dv) src[s][jj][kk][c]      (exact transpose of the Joseph forward, S9; w_s applied later)
template <int D>
__device__ __forceinline__ void gather_voxel(const TcProj &pg, const float *__restrict__ src_s, int x, int y, int z,
                                             int J, int Kd, float (&t)[D])
{
#pragma unroll
    for (int c = 0; c < D; c++) t[c] = 0.f;
    const double j0 = fma((double)x, pg.Jx0, fma((double)y, pg.Jx1, fma((double)z, pg.Jx2, pg.Jc)));
    const double k0 = fma((double)x, pg.Kx0, fma((double)y, pg.Kx1, fma((double)z, pg.Kx2, pg.Kc)));
    const double fj0 = floor(j0), fk0 = floor(k0);
    const int jb = (int)fj0, kb = (int)fk0;
    const float fj = (float)(j0 - fj0), fk = (float)(k0 - fk0);
    const int djlo = max((int)ceilf(fj - pg.hj), -jb), djhi = min((int)floorf(fj + pg.hj), J - 1 - jb);
    const int dklo = max((int)ceilf(fk - pg.hk), -kb), dkhi = min((int)floorf(fk + pg.hk), Kd - 1 - kb);
    for (int dj = djlo; dj <= djhi; dj++) {
        const float ej = (float)dj - fj;
        const float au = pg.mju * ej, av = pg.mjv * ej;
        const float *row = src_s + ((long long)(jb + dj) * Kd + kb) * D;
        for (int dk = dklo; dk <= dkhi; dk++) {
            const float ek = (float)dk - fk;
            const float du = fmaf(pg.mku, ek, au), dv = fmaf(pg.mkv, ek, av);
            const float wt = fmaxf(0.f, 1.f - fabsf(du)) * fmaxf(0.f, 1.f - fabsf(dv));
            if (wt > 0.f) {
                const float4 *p = reinterpret_cast<const float4 *>(row + dk * D);
#pragma unroll
                for (int c = 0; c < D; c += 4) {
                    const float4 r = __ldg(p + c / 4);
                    t[c] = fmaf(wt, r.x, t[c]); t[c + 1] = fmaf(wt, r.y, t[c + 1]);
                    t[c + 2] = fmaf(wt, r.z, t[c + 2]); t[c + 3] = fmaf(wt, r.w, t[c + 3]);
                }
            }
        }
    }
}

// Fast path of gather_voxel for candidate windows at most 3 rays wide (hj, hk < 1.5: every projection of the
// standard geometry, where hj, hk <= sqrt 2): the 3 x 3 candidates are evaluated branch-free with fixed
// offsets, so their loads are independent and overlap; rays outside the detector or with zero weight are
// predicated off.  Same weights as gather_voxel.
template <int D>
__device__ __forceinline__ void gather_voxel3(const TcProj &pg, const float *__restrict__ src_s, int x, int y, int z,
                                              int J, int Kd, float (&t)[D])
{
#pragma unroll
    for (int c = 0; c < D; c++) t[c] = 0.f;
    const double j0 = fma((double)x, pg.Jx0, fma((double)y, pg.Jx1, fma((double)z, pg.Jx2, pg.Jc)));
    const double k0 = fma((double)x, pg.Kx0, fma((double)y, pg.Kx1, fma((double)z, pg.Kx2, pg.Kc)));
    const int jb = __double2int_rd(j0), kb = __double2int_rd(k0);
    const float fj = (float)(j0 - (double)jb), fk = (float)(k0 - (double)kb);
    const int dj0 = (int)ceilf(fj - pg.hj), dk0 = (int)ceilf(fk - pg.hk);
    const int jj0 = jb + dj0, kk0 = kb + dk0;
    float au[3], av[3], bu[3], bv[3];
    bool rok[3], cok[3];
#pragma unroll
    for (int r = 0; r < 3; r++) {
        const float ej = (float)(dj0 + r) - fj, ek = (float)(dk0 + r) - fk;
        au[r] = pg.mju * ej; av[r] = pg.mjv * ej;
        bu[r] = pg.mku * ek; bv[r] = pg.mkv * ek;
        rok[r] = (unsigned)(jj0 + r) < (unsigned)J;
        cok[r] = (unsigned)(kk0 + r) < (unsigned)Kd;
    }
    const float *p00 = src_s + ((long long)jj0 * Kd + kk0) * D;
#pragma unroll
    for (int r = 0; r < 3; r++) {
        const float *row = p00 + (long long)r * Kd * D;
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const float du = au[r] + bu[c], dv = av[r] + bv[c];
            const float wt = fmaxf(0.f, 1.f - fabsf(du)) * fmaxf(0.f, 1.f - fabsf(dv));
            if (wt > 0.f && rok[r] && cok[c]) {
                const float4 *p = reinterpret_cast<const float4 *>(row + c * D);
#pragma unroll
                for (int q = 0; q < D; q += 4) {
                    const float4 v = __ldg(p + q / 4);
                    t[q] = fmaf(wt, v.x, t[q]); t[q + 1] = fmaf(wt, v.y, t[q + 1]);
                    t[q + 2] = fmaf(wt, v.z, t[q + 2]); t[q + 3] = fmaf(wt, v.w, t[q + 3]);
                }
            }
        }
    }
}

// two accumulators of ACCW columns each (ping-pong between accumulation windows)
template <int NPAD>
struct TcCols {
    static constexpr int accw = NPAD <= 16 ? 16 : (NPAD <= 32 ? 32 : 64);
    static constexpr int value = 2 * accw < 32 ? 32 : 2 * accw;
};

template <int D, int NPAD>
__global__ void __launch_bounds__(TC_THREADS, 4) adjoint_tc_kernel(const AdjArgs a)
{
    constexpr int KC = (D <= 16) ? 16 : D;        // contraction columns per stage
    constexpr int NPC = KC / D;                   // projections per stage
    constexpr int A_FLOATS = TC_M * KC, B_FLOATS = NPAD * KC;
    constexpr int TCOLS = TcCols<NPAD>::value, ACCW = TcCols<NPAD>::accw;
    constexpr int WIN = 8;                        // chunks per accumulation window (see flush_window)
    constexpr uint32_t IDESC = idesc_tf32(TC_M, NPAD);
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    float *sA = reinterpret_cast<float *>(smem_raw);                  // [stage][hi,lo][A_FLOATS]
    float *sB = sA + 4 * A_FLOATS;                                    // [stage][hi,lo][B_FLOATS]
    TcProj *sp = reinterpret_cast<TcProj *>(sB + 4 * B_FLOATS);       // [2][NPC]
    uint64_t *mbar = reinterpret_cast<uint64_t *>(sp + 2 * NPC);      // [2] stage free, [2] window complete
    uint64_t *wbar = mbar + 2;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(mbar + 4);

    const int tid = threadIdx.x, warp = tid >> 5;
    const long long nvox = (long long)a.X * a.Y * a.Z;
    const long long vox = (long long)blockIdx.x * TC_M + tid;
    const bool ok = vox < nvox;
    const long long vv = ok ? vox : nvox - 1;
    const int z = (int)(vv % a.Z), y = (int)((vv / a.Z) % a.Y), x = (int)(vv / ((long long)a.Z * a.Y));
    const long long proj_stride = (long long)a.J * a.Kd * D;

    if (warp == 0) tmem_alloc<TCOLS>(tmem_slot);
    if (tid == 0) {
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        mbar_init(&wbar[0], 1);
        mbar_init(&wbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid < NPC) load_proj(sp[tid], a.tab, tid, a.P);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_acc = *tmem_slot;

    // The tensor core adds into its fp32 accumulator with truncation (measured: a systematic -3e-8 relative
    // shrink per accumulation, -1.6e-5 over the 1080 MMAs of config 5), so accumulation is cut into windows of
    // WIN chunks that alternate between two TMEM accumulators; a finished window is drained into registers
    // and summed there in round-to-nearest fp32 while the next window is already running.
    float racc[NPAD];
#pragma unroll
    for (int i = 0; i < NPAD; i++) racc[i] = 0.f;
    auto flush_window = [&](int w) {
        mbar_wait(&wbar[w & 1], (uint32_t)((w >> 1) & 1));
        tc_fence_after();
#pragma unroll
        for (int c0 = 0; c0 < NPAD; c0 += 16) {
            float v[16];
            tmem_ld16(tmem_acc + ((uint32_t)(warp * 32) << 16) + (uint32_t)((w & 1) * ACCW + c0), v);
#pragma unroll
            for (int i = 0; i < 16; i++) racc[c0 + i] += v[i];
        }
    };

    const int nch = (a.P + NPC - 1) / NPC;
    for (int ch = 0; ch < nch; ch++) {
        const int st = ch & 1, s0 = ch * NPC;
        if (ch >= 2) mbar_wait(&mbar[st], (uint32_t)(((ch >> 1) - 1) & 1));   // MMAs of chunk ch-2 have read stage st
        if (ch >= WIN && ch % WIN == 1) flush_window(ch / WIN - 1);             // its MMAs had a whole chunk to finish
        float *Ahi = sA + (2 * st) * A_FLOATS, *Alo = Ahi + A_FLOATS;
        float *Bhi = sB + (2 * st) * B_FLOATS, *Blo = Bhi + B_FLOATS;
        // prefetch the next chunk's projection constants (read after this chunk's barrier)
        if (tid < NPC) load_proj(sp[(st ^ 1) * NPC + tid], a.tab, s0 + NPC + tid, a.P);
        // B operand: element (n = channel i, k = (p, c)) = w_s B[s0+p][i][c], split hi/lo
        for (int g = tid; g < NPAD * (KC / 4); g += TC_THREADS) {
            const int n = g % NPAD, kg = g / NPAD;                    // 16-byte group: columns 4kg .. 4kg+3
            const int p = (4 * kg) / D, c = (4 * kg) % D, s = s0 + p;
            float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
            if (n < a.K && s < a.P) {
                b = __ldg(reinterpret_cast<const float4 *>(a.B + ((long long)s * a.K + n) * D + c));
                const float w = a.tab[s].w;
                b.x *= w; b.y *= w; b.z *= w; b.w *= w;
            }
            float4 h, l;
            split_tf32(b.x, h.x, l.x); split_tf32(b.y, h.y, l.y); split_tf32(b.z, h.z, l.z); split_tf32(b.w, h.w, l.w);
            *reinterpret_cast<float4 *>(Bhi + kg * (NPAD * 4) + n * 4) = h;
            *reinterpret_cast<float4 *>(Blo + kg * (NPAD * 4) + n * 4) = l;
        }
        // A operand: this thread's row = its voxel's gathered D-channel values for the chunk's projections
#pragma unroll
        for (int p = 0; p < NPC; p++) {
            float t[D];
            const TcProj &pg = sp[st * NPC + p];
            const float *src_s = a.src + (long long)min(s0 + p, a.P - 1) * proj_stride;
            if (pg.valid == 2) gather_voxel3<D>(pg, src_s, x, y, z, a.J, a.Kd, t);
            else gather_voxel<D>(pg, src_s, x, y, z, a.J, a.Kd, t);
#pragma unroll
            for (int c = 0; c < D; c += 4) {
                const int kg = (p * D + c) / 4;
                float4 h, l;
                split_tf32(ok ? t[c] : 0.f, h.x, l.x); split_tf32(ok ? t[c + 1] : 0.f, h.y, l.y);
                split_tf32(ok ? t[c + 2] : 0.f, h.z, l.z); split_tf32(ok ? t[c + 3] : 0.f, h.w, l.w);
                *reinterpret_cast<float4 *>(Ahi + kg * (TC_M * 4) + tid * 4) = h;
                *reinterpret_cast<float4 *>(Alo + kg * (TC_M * 4) + tid * 4) = l;
            }
        }
        fence_async_smem();
        tc_fence_before();
        __syncthreads();
        if (tid == 0) {
            tc_fence_after();
            const uint32_t a_hi = smem_u32(Ahi), a_lo = smem_u32(Alo), b_hi = smem_u32(Bhi), b_lo = smem_u32(Blo);
#pragma unroll
            for (int ks = 0; ks < KC / 8; ks++) {
                const uint32_t ao = ks * 2 * (TC_M * 16), bo = ks * 2 * (NPAD * 16);
                const uint64_t dAh = smem_desc(a_hi + ao, TC_M * 16, 128), dAl = smem_desc(a_lo + ao, TC_M * 16, 128);
                const uint64_t dBh = smem_desc(b_hi + bo, NPAD * 16, 128), dBl = smem_desc(b_lo + bo, NPAD * 16, 128);
                const uint32_t acc = tmem_acc + (uint32_t)(((ch / WIN) & 1) * ACCW);
                mma_tf32(acc, dAl, dBh, IDESC, ((ch % WIN) | ks) ? 1u : 0u);      // small terms first
                mma_tf32(acc, dAh, dBl, IDESC, 1u);
                mma_tf32(acc, dAh, dBh, IDESC, 1u);
            }
            tc_commit(&mbar[st]);
            if (ch % WIN == WIN - 1 || ch == nch - 1) tc_commit(&wbar[(ch / WIN) & 1]);
        }
    }
    // epilogue: drain the windows still in tensor memory, then registers -> grad (thread = voxel row)
    {
        const int nwin = (nch + WIN - 1) / WIN;
        if (nwin >= 2 && (nch - 1) % WIN == 0) flush_window(nwin - 2);     // the loop had not reached its flush point
        flush_window(nwin - 1);
        if (ok) {
            float *o = a.out + vox * a.ldk;
#pragma unroll
            for (int c = 0; c < NPAD; c += 4)
                if (c < a.ldk)                      // ldk % 4 == 0 on this path
                    *reinterpret_cast<float4 *>(o + c) = make_float4(racc[c], racc[c + 1], racc[c + 2], racc[c + 3]);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<TCOLS>(tmem_acc);
}

template <int D, int NPAD>
cudaError_t launch_tc(const AdjArgs &a, cudaStream_t st)
{
    constexpr int KC = (D <= 16) ? 16 : D;
    constexpr int NPC = KC / D;
    const size_t smem = (size_t)4 * (TC_M * KC + NPAD * KC) * sizeof(float) + 2 * NPC * sizeof(TcProj) + 4 * sizeof(uint64_t) + 16;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(adjoint_tc_kernel<D, NPAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    const long long nvox = (long long)a.X * a.Y * a.Z;
    adjoint_tc_kernel<D, NPAD><<<(unsigned)((nvox + TC_M - 1) / TC_M), TC_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

}  // namespace

bool mm_adjoint_tc_supported(const AdjArgs &a)
{
    return a.vec_ok && (a.D == 8 || a.D == 16) && a.ldk % 4 == 0 && a.ldk <= 64 &&
           (reinterpret_cast<uintptr_t>(a.B) & 15u) == 0 && (reinterpret_cast<uintptr_t>(a.out) & 15u) == 0;
}

int mm_adjoint_tc_launch(const AdjArgs &a, void *stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    const int npad = (a.ldk + 15) / 16 * 16;
    if (a.D == 8) {
        if (npad == 16) return launch_tc<8, 16>(a, st);
        if (npad == 32) return launch_tc<8, 32>(a, st);
        if (npad == 48) return launch_tc<8, 48>(a, st);
        return launch_tc<8, 64>(a, st);
    }
    if (npad == 16) return launch_tc<16, 16>(a, st);
    if (npad == 32) return launch_tc<16, 32>(a, st);
    if (npad == 48) return launch_tc<16, 48>(a, st);
    return launch_tc<16, 64>(a, st);
}
