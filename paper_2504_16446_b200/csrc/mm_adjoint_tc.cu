// mm_adjoint_tc.cu — fused adjoint A^T (steps a6 + a7) with the basis contraction on the 5th-gen tensor cores.
//
//   grad[x][i] = sum_s sum_c  ( w_s B[s][i][c] ) * t[x][s][c],      t[x][s][c] = sum_(j,k) Lambda Lambda wr[s][j][k][c]
//
// The gather t (exact transpose of the Joseph forward, reading S9) is irregular and stays on the
// CUDA cores, one thread per voxel.  The contraction over (s,c) is a dense GEMM  [128 voxels x (P*D)] . [(P*D) x ldk]
// (2.17 T FMA on BASELINE config 5, the adjoint's dominant term): each CTA streams its
// 128 x 16 slices of t through shared memory into tcgen05.mma (kind::tf32, M=128, N=ldk, K=8) with the fp32
// accumulators in tensor memory.  Plain TF32 (10-bit mantissa) cannot meet the 1e-5 parity bar, so both operands
// are split x = hi + lo with hi = x rounded to TF32 and lo = x - hi (exact), and three products are issued:
// lo*hi + hi*lo + hi*hi (error ~2^-21 per term).  The MMA's fp32 accumulation truncates, so it is cut into
// windows that are summed in round-to-nearest fp32 (see drain_window).
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
constexpr int TC_THREADS = 160;      // 4 gather warps + 1 operand/MMA warp
#ifndef TC_MINB
#define TC_MINB 4
#endif

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

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const float (&v)[16])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
        ::"r"(taddr), "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])),
          "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])),
          "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])), "r"(__float_as_uint(v[11])),
          "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])), "r"(__float_as_uint(v[15]))
        : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

// x = hi + lo: hi = x rounded to nearest TF32 (1+8+10 bits), lo = x - hi exactly (|lo| <= 2^-11 |x|, either
// sign).  The tensor core ignores the 13 low mantissa bits of lo (error <= 2^-21 |x|, unbiased because of lo's
// random sign); truncating hi instead of rounding it makes lo one-signed and the error a bias (measured).
__device__ __forceinline__ void split_tf32(float x, float &hi, float &lo)
{
    uint32_t h;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(h) : "f"(x));
    hi = __uint_as_float(h);
    lo = x - hi;
}

// the gather block of MMProj (same 96-byte layout, checked below)
struct TcProj {
    double Jc, Jx0, Jx1, Jx2, Kc, Kx0, Kx1, Kx2;
    float mju, mku, mjv, mkv, hj, hk, w;
    int valid;                     // MMProj::gcode, or 0 for a projection past the last one
};
static_assert(sizeof(TcProj) == 96, "TcProj mirrors the gather block of MMProj");

// 12 lanes copy one projection's constants (8 bytes each) from the device table into shared memory
__device__ __forceinline__ void load_proj(TcProj *dst, const MMProj *tab, int s, int P, int word)
{
    uint2 v = make_uint2(0u, 0u);                  // past the end: all zero, valid = 0
    if (s < P) v = __ldg(reinterpret_cast<const uint2 *>(&tab[s].Jc) + word);
    reinterpret_cast<uint2 *>(dst)[word] = v;
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

// v[0..7] = on ? 32 bytes at p : 0 — a predicated read-only 256-bit load (sm_100: LDG.E.256), no branch;
// p must be 32-byte aligned when on
__device__ __forceinline__ void ldg256_pred(const void *p, bool on, float *v)
{
#pragma unroll
    for (int i = 0; i < 8; i++) v[i] = 0.f;
    asm volatile(
        "{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %9, 0;\n\t"
        "@q ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n\t}"
        : "+f"(v[0]), "+f"(v[1]), "+f"(v[2]), "+f"(v[3]), "+f"(v[4]), "+f"(v[5]), "+f"(v[6]), "+f"(v[7])
        : "l"(p), "r"((int)on));
}

// Fast path of gather_voxel for candidate windows NJ x NK rays wide, NJ, NK in {2, 3}: hj <= 1 means at most two
// candidate rows (|dj - fj| < hj), hj < 1.5 at most three (every projection of the standard geometry has
// hj, hk <= sqrt 2; on config 5, 44 % / 87 % of the projections have hj / hk <= 1, 5.4 candidates on average
// instead of 9).  Candidates are evaluated at fixed offsets; rays outside the detector or with zero weight
// are skipped.  Same weights as gather_voxel.
template <int D, int NJ, int NK>
__device__ __forceinline__ void gather_voxel_fixed(const TcProj &pg, const float *__restrict__ src_s, int x, int y, int z,
                                                   int J, int Kd, float (&t)[D])
{
#pragma unroll
    for (int c = 0; c < D; c++) t[c] = 0.f;
    const double j0 = fma((double)x, pg.Jx0, fma((double)y, pg.Jx1, fma((double)z, pg.Jx2, pg.Jc)));
    const double k0 = fma((double)x, pg.Kx0, fma((double)y, pg.Kx1, fma((double)z, pg.Kx2, pg.Kc)));
    const int jb = __double2int_rd(j0), kb = __double2int_rd(k0);
    const float fj = (float)(j0 - (double)jb), fk = (float)(k0 - (double)kb);
    // first candidate: smallest integer above f - h (h capped at 1 for a 2-wide window: exactly-1 half-widths
    // carry 2e-6 of slack in the table)
    const int dj0 = (int)ceilf(fj - (NJ == 2 ? fminf(pg.hj, 1.f) : pg.hj));
    const int dk0 = (int)ceilf(fk - (NK == 2 ? fminf(pg.hk, 1.f) : pg.hk));
    const int jj0 = jb + dj0, kk0 = kb + dk0;
    float au[NJ], av[NJ], bu[NK], bv[NK];
    bool rok[NJ], cok[NK];
#pragma unroll
    for (int r = 0; r < NJ; r++) {
        const float ej = (float)(dj0 + r) - fj;
        au[r] = pg.mju * ej; av[r] = pg.mjv * ej;
        rok[r] = (unsigned)(jj0 + r) < (unsigned)J;
    }
#pragma unroll
    for (int c = 0; c < NK; c++) {
        const float ek = (float)(dk0 + c) - fk;
        bu[c] = pg.mku * ek; bv[c] = pg.mkv * ek;
        cok[c] = (unsigned)(kk0 + c) < (unsigned)Kd;
    }
    // 32-bit float4 index into the projection's sinogram (J*Kd*D < 2^31 checked by the host)
    const float4 *src4 = reinterpret_cast<const float4 *>(src_s);
    const int i00 = (jj0 * Kd + kk0) * (D / 4), rstep = Kd * (D / 4);
    // all candidates' loads are issued (predicated, branch-free) before the first FMA: one memory round trip per
    // voxel-projection instead of one per candidate
    float wt[NJ * NK], v[NJ * NK][D];
#pragma unroll
    for (int r = 0; r < NJ; r++) {
#pragma unroll
        for (int c = 0; c < NK; c++) {
            const float du = au[r] + bu[c], dv = av[r] + bv[c];
            const float w = fmaxf(0.f, 1.f - fabsf(du)) * fmaxf(0.f, 1.f - fabsf(dv));
            const bool on = w > 0.f && rok[r] && cok[c];
            wt[r * NK + c] = on ? w : 0.f;
            const float4 *p = src4 + (i00 + r * rstep + c * (D / 4));
#pragma unroll
            for (int q = 0; q < D; q += 8) ldg256_pred(p + q / 4, on, &v[r * NK + c][q]);
        }
    }
#pragma unroll
    for (int n = 0; n < NJ * NK; n++)
#pragma unroll
        for (int i = 0; i < D; i++) t[i] = fmaf(wt[n], v[n][i], t[i]);
}

// The paper's own adjoint ("bilinear interpolation of the projection"; NEXT-1): the four pixels
// around the voxel's detector position with weights (1-fj | fj)(1-fk | fk); pixels off the detector count as 0.
template <int D>
__device__ __forceinline__ void gather_voxel_bilinear(const TcProj &pg, const float *__restrict__ src_s, int x, int y, int z,
                                                      int J, int Kd, float (&t)[D])
{
#pragma unroll
    for (int c = 0; c < D; c++) t[c] = 0.f;
    const double j0 = fma((double)x, pg.Jx0, fma((double)y, pg.Jx1, fma((double)z, pg.Jx2, pg.Jc)));
    const double k0 = fma((double)x, pg.Kx0, fma((double)y, pg.Kx1, fma((double)z, pg.Kx2, pg.Kc)));
    const int jb = __double2int_rd(j0), kb = __double2int_rd(k0);
    const float fj = (float)(j0 - (double)jb), fk = (float)(k0 - (double)kb);
    const float4 *src4 = reinterpret_cast<const float4 *>(src_s);
    const int i00 = (jb * Kd + kb) * (D / 4), rstep = Kd * (D / 4);
    float wt[4], v[4][D];
#pragma unroll
    for (int r = 0; r < 2; r++) {
#pragma unroll
        for (int c = 0; c < 2; c++) {
            const bool on = (unsigned)(jb + r) < (unsigned)J && (unsigned)(kb + c) < (unsigned)Kd;
            wt[2 * r + c] = (r ? fj : 1.f - fj) * (c ? fk : 1.f - fk);
            const float4 *p = src4 + (i00 + r * rstep + c * (D / 4));
#pragma unroll
            for (int q = 0; q < D; q += 8) ldg256_pred(p + q / 4, on, &v[2 * r + c][q]);
        }
    }
#pragma unroll
    for (int n = 0; n < 4; n++)
#pragma unroll
        for (int i = 0; i < D; i++) t[i] = fmaf(wt[n], v[n][i], t[i]);
}

// two regions of ACCW columns each: the MMA accumulator of the current window, and the running sum
template <int NPAD>
struct TcCols {
    static constexpr int accw = NPAD <= 16 ? 16 : (NPAD <= 32 ? 32 : (NPAD <= 64 ? 64 : (NPAD <= 128 ? 128 : 256)));
    static constexpr int value = 2 * accw < 32 ? 32 : 2 * accw;      // a power of two, at most 512
};

__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// Warp roles: warps 0-3 gather (thread = voxel = operand row = TMEM lane); warp 4 stages the B operand and issues
// the MMAs.  No block-wide barrier inside the projection loop: a gather thread arrives on full[stage] when its
// row is in shared memory, the MMA thread waits for all 128 arrivals, and tcgen05.commit releases the stage
// through empty[stage], so a slow warp delays only the MMA, not the other warps' loads.
template <int D, int NPAD>
__global__ void __launch_bounds__(TC_THREADS, TC_MINB) adjoint_tc_kernel(const AdjArgs a)
{
    constexpr int KC = (D <= 16) ? 16 : D;        // contraction columns per stage
    constexpr int NPC = KC / D;                   // projections per stage
    constexpr int A_FLOATS = TC_M * KC, B_FLOATS = NPAD * KC;
    constexpr int TCOLS = TcCols<NPAD>::value, ACCW = TcCols<NPAD>::accw;
    constexpr int WIN = 8;                        // chunks per accumulation window (see drain_window)
    constexpr uint32_t IDESC = idesc_tf32(TC_M, NPAD);
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    float *sA = reinterpret_cast<float *>(smem_raw);                  // [stage][hi,lo][A_FLOATS]
    float *sB = sA + 4 * A_FLOATS;                                    // [stage][hi,lo][B_FLOATS]
    TcProj *sp = reinterpret_cast<TcProj *>(sB + 4 * B_FLOATS);       // [4 gather warps][NPC] private copies
    uint64_t *full = reinterpret_cast<uint64_t *>(sp + 4 * NPC);      // [2] rows of the stage written
    uint64_t *empty = full + 2;                                       // [2] MMAs have read the stage
    uint64_t *wbar = full + 4;                                        // MMAs of an accumulation window complete
    uint64_t *drained = full + 5;                                     // all rows of the window added to the running sum
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(full + 6);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int nch = (a.P + NPC - 1) / NPC;

    if (warp == 4) tmem_alloc<TCOLS>(tmem_slot);
    if (tid == 0) {
        mbar_init(&full[0], TC_M); mbar_init(&full[1], TC_M);
        mbar_init(&empty[0], 1); mbar_init(&empty[1], 1);
        mbar_init(wbar, 1); mbar_init(drained, TC_M);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_acc = *tmem_slot;

    if (warp == 4) {
        // ---------------- B operand + MMA issue ----------------
        // element (n = channel i, k = (p, c)) of a stage's B tile = w_s B[s0+p][i][c]; its NPAD*KC/4 16-byte
        // groups are spread over the 32 lanes.  The global loads for chunk ch+1 are issued before this warp
        // waits for chunk ch's rows, so their latency is off the MMA's critical path.
        constexpr int BG = (NPAD * (KC / 4) + 31) / 32;       // groups per lane
        constexpr bool PREFETCH_B = BG <= 8;                  // wide accumulators: load B in place instead
        float4 breg[PREFETCH_B ? BG : 1];
        auto fetch_b = [&](int g, int s0) -> float4 {
            const int n = g % NPAD, kg = g / NPAD;                    // 16-byte group: columns 4kg .. 4kg+3
            const int p = (4 * kg) / D, c = (4 * kg) % D, s = s0 + p;
            float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
            if (g < NPAD * (KC / 4) && n < a.K && s < a.P) {
                b = __ldg(reinterpret_cast<const float4 *>(a.B + ((long long)s * a.K + n) * D + c));
                const float w = __ldg(&a.tab[s].w);
                b.x *= w; b.y *= w; b.z *= w; b.w *= w;
            }
            return b;
        };
        auto store_b = [&](int g, const float4 &b, float *Bhi, float *Blo) {
            const int n = g % NPAD, kg = g / NPAD;
            float4 h, l;
            split_tf32(b.x, h.x, l.x); split_tf32(b.y, h.y, l.y); split_tf32(b.z, h.z, l.z); split_tf32(b.w, h.w, l.w);
            *reinterpret_cast<float4 *>(Bhi + kg * (NPAD * 4) + n * 4) = h;
            *reinterpret_cast<float4 *>(Blo + kg * (NPAD * 4) + n * 4) = l;
        };
        if constexpr (PREFETCH_B) {
#pragma unroll
            for (int i = 0; i < BG; i++) breg[i] = fetch_b(lane + 32 * i, 0);
        }
        for (int ch = 0; ch < nch; ch++) {
            const int st = ch & 1;
            if (ch >= 2) mbar_wait(&empty[st], (uint32_t)(((ch >> 1) - 1) & 1));
            float *Bhi = sB + (2 * st) * B_FLOATS, *Blo = Bhi + B_FLOATS;
            if constexpr (PREFETCH_B) {
#pragma unroll
                for (int i = 0; i < BG; i++)
                    if (lane + 32 * i < NPAD * (KC / 4)) store_b(lane + 32 * i, breg[i], Bhi, Blo);
                if (ch + 1 < nch) {
#pragma unroll
                    for (int i = 0; i < BG; i++) breg[i] = fetch_b(lane + 32 * i, (ch + 1) * NPC);
                }
            } else {
                for (int g = lane; g < NPAD * (KC / 4); g += 32) store_b(g, fetch_b(g, ch * NPC), Bhi, Blo);
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) {
                mbar_wait(&full[st], (uint32_t)((ch >> 1) & 1));
                tc_fence_after();
                const float *Ahi = sA + (2 * st) * A_FLOATS;
                const uint32_t a_hi = smem_u32(Ahi), a_lo = smem_u32(Ahi + A_FLOATS), b_hi = smem_u32(Bhi), b_lo = smem_u32(Blo);
                const uint32_t acc = tmem_acc;
                if (ch >= WIN && ch % WIN == 0) {          // the previous window must have left the accumulator
                    mbar_wait(drained, (uint32_t)((ch / WIN - 1) & 1));
                    tc_fence_after();
                }
#pragma unroll
                for (int ks = 0; ks < KC / 8; ks++) {
                    const uint32_t ao = ks * 2 * (TC_M * 16), bo = ks * 2 * (NPAD * 16);
                    const uint64_t dAh = smem_desc(a_hi + ao, TC_M * 16, 128), dAl = smem_desc(a_lo + ao, TC_M * 16, 128);
                    const uint64_t dBh = smem_desc(b_hi + bo, NPAD * 16, 128), dBl = smem_desc(b_lo + bo, NPAD * 16, 128);
                    mma_tf32(acc, dAl, dBh, IDESC, ((ch % WIN) | ks) ? 1u : 0u);      // small terms first
                    mma_tf32(acc, dAh, dBl, IDESC, 1u);
                    mma_tf32(acc, dAh, dBh, IDESC, 1u);
                }
                tc_commit(&empty[st]);
                if (ch % WIN == WIN - 1 || ch == nch - 1) tc_commit(wbar);
            }
            __syncwarp();
        }
    } else {
        // ---------------- gather warps ----------------
        const long long nvox = a.vox_end;
        const long long vox = a.vox_begin + (long long)blockIdx.x * TC_M + tid;
        const bool ok = vox < nvox;
        const long long vv = ok ? vox : nvox - 1;
        const int z = (int)(vv % a.Z), y = (int)((vv / a.Z) % a.Y), x = (int)(vv / ((long long)a.Z * a.Y));
        const long long proj_stride = (long long)a.J * a.Kd * D;
        TcProj *wsp = sp + warp * NPC;

        // The tensor core adds into its fp32 accumulator with truncation (measured: a systematic -3e-8 relative
        // shrink per accumulation, -1.6e-5 over the 1080 MMAs of config 5), so accumulation is cut into windows
        // of WIN chunks: when a window's MMAs are complete every thread adds its row of the accumulator to a
        // running sum in round-to-nearest fp32.  The running sum lives in tensor memory too (columns ACCW..),
        // so it costs no registers between windows.
        const uint32_t lane_base = tmem_acc + ((uint32_t)(warp * 32) << 16);
        auto drain_window = [&](int w) {
            mbar_wait(wbar, (uint32_t)(w & 1));
            tc_fence_after();
#pragma unroll
            for (int c0 = 0; c0 < NPAD; c0 += 16) {
                float v[16];
                tmem_ld16(lane_base + c0, v);
                if (w > 0) {
                    float m[16];
                    tmem_ld16(lane_base + ACCW + c0, m);
#pragma unroll
                    for (int i = 0; i < 16; i++) v[i] += m[i];
                }
                tmem_st16(lane_base + ACCW + c0, v);
            }
            tc_fence_before();
            mbar_arrive(drained);
        };

        for (int ch = 0; ch < nch; ch++) {
            const int st = ch & 1, s0 = ch * NPC;
            __syncwarp();
            if (lane < 12 * NPC) load_proj(wsp + lane / 12, a.tab, s0 + lane / 12, a.P, lane % 12);   // this warp's copy
            __syncwarp();
            if (ch >= 2) mbar_wait(&empty[st], (uint32_t)(((ch >> 1) - 1) & 1));   // MMAs of chunk ch-2 have read stage st
            float *Ahi = sA + (2 * st) * A_FLOATS, *Alo = Ahi + A_FLOATS;
#pragma unroll 1                     // one projection's nine 256-bit loads in flight is what the register file holds
            for (int p = 0; p < NPC; p++) {
                float t[D];
                const TcProj &pg = wsp[p];
                const float *src_s = a.src + (long long)min(s0 + p, a.P - 1) * proj_stride;
                if (a.bilinear) {
                    if (pg.valid) gather_voxel_bilinear<D>(pg, src_s, x, y, z, a.J, a.Kd, t);
                    else {
#pragma unroll
                        for (int c = 0; c < D; c++) t[c] = 0.f;
                    }
                } else
                switch (pg.valid) {                                   // uniform across the block
                    case 4: gather_voxel_fixed<D, 2, 2>(pg, src_s, x, y, z, a.J, a.Kd, t); break;
                    case 5: gather_voxel_fixed<D, 2, 3>(pg, src_s, x, y, z, a.J, a.Kd, t); break;
                    case 6: gather_voxel_fixed<D, 3, 2>(pg, src_s, x, y, z, a.J, a.Kd, t); break;
                    case 7: gather_voxel_fixed<D, 3, 3>(pg, src_s, x, y, z, a.J, a.Kd, t); break;
                    case 0:
#pragma unroll
                        for (int c = 0; c < D; c++) t[c] = 0.f;
                        break;
                    default: gather_voxel<D>(pg, src_s, x, y, z, a.J, a.Kd, t); break;
                }
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
            mbar_arrive(&full[st]);
            if (ch % WIN == WIN - 1 || ch == nch - 1) drain_window(ch / WIN);
        }
        // epilogue: running sum (thread = voxel row) -> grad
        float *o = a.out + vox * a.ldk;
#pragma unroll
        for (int c0 = 0; c0 < NPAD; c0 += 16) {
            float v[16];
            tmem_ld16(lane_base + ACCW + c0, v);
            if (ok) {
#pragma unroll
                for (int i = 0; i < 16; i += 4)
                    if (c0 + i < a.ldk)             // ldk % 4 == 0 on this path
                        *reinterpret_cast<float4 *>(o + c0 + i) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 4) tmem_dealloc<TCOLS>(tmem_acc);
}

template <int D, int NPAD>
cudaError_t launch_tc(const AdjArgs &a, cudaStream_t st)
{
    constexpr int KC = (D <= 16) ? 16 : D;
    constexpr int NPC = KC / D;
    const size_t smem = (size_t)4 * (TC_M * KC + NPAD * KC) * sizeof(float) + 4 * NPC * sizeof(TcProj) + 6 * sizeof(uint64_t) + 16;
    // every launch: the attribute is per device (a process-wide "configured" flag breaks the second device) and the
    // call costs a few hundred nanoseconds
    const cudaError_t e = cudaFuncSetAttribute(adjoint_tc_kernel<D, NPAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long nvox = a.vox_end - a.vox_begin;
    if (nvox <= 0) return cudaSuccess;
    adjoint_tc_kernel<D, NPAD><<<(unsigned)((nvox + TC_M - 1) / TC_M), TC_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

}  // namespace

bool mm_adjoint_tc_supported(const AdjArgs &a)
{
    return a.vec_ok && (a.D == 8 || a.D == 16) && a.ldk % 4 == 0 && a.ldk <= 256 &&
           (long long)a.J * a.Kd * a.D < (1LL << 31) &&
           (reinterpret_cast<uintptr_t>(a.B) & 15u) == 0 && (reinterpret_cast<uintptr_t>(a.out) & 15u) == 0 &&
           (reinterpret_cast<uintptr_t>(a.src) & 31u) == 0;      // 256-bit gather loads
}

int mm_adjoint_tc_launch(const AdjArgs &a, void *stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    // accumulator width: the smallest instantiated multiple of 16 that holds ldk channels
    const int w = a.ldk <= 16 ? 16 : a.ldk <= 32 ? 32 : a.ldk <= 48 ? 48 : a.ldk <= 64 ? 64 : a.ldk <= 96 ? 96 : a.ldk <= 128 ? 128
                : a.ldk <= 192 ? 192 : 256;
#define MM_TC_CASE(DD, NN) if (a.D == DD && w == NN) return launch_tc<DD, NN>(a, st)
    MM_TC_CASE(8, 16); MM_TC_CASE(8, 32); MM_TC_CASE(8, 48); MM_TC_CASE(8, 64);
    MM_TC_CASE(8, 96); MM_TC_CASE(8, 128); MM_TC_CASE(8, 192); MM_TC_CASE(8, 256);
    MM_TC_CASE(16, 16); MM_TC_CASE(16, 32); MM_TC_CASE(16, 48); MM_TC_CASE(16, 64);
    MM_TC_CASE(16, 96); MM_TC_CASE(16, 128); MM_TC_CASE(16, 192); MM_TC_CASE(16, 256);
#undef MM_TC_CASE
    return cudaErrorInvalidValue;
}
