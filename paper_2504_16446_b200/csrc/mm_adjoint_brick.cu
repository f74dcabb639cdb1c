// mm_adjoint_brick.cu — fused adjoint A^T (steps a6 + a7), the primary path of mm_adjoint / phase 2 of mm_loss_gradient.
//
//   grad[x][i] = sum_s sum_c  ( w_s B[s][i][c] ) * t[x][s][c],      t[x][s][c] = sum_(j,k) Lambda(du) Lambda(dv) wr[s][j][k][c]
//
// (exact transpose of the Joseph forward, reading S9; with the identity in place of M and a 2 x 2
// window the same code is the paper's bilinear back-projector, NEXT-1.)
//
// Design (B200):
//  * A CTA owns a BRICK of 4 x 4 x 8 = 128 voxels (thread = voxel = accumulator row = TMEM lane).  A brick's shadow on
//    the detector is compact (<= 13 x 13 pixels in the standard geometry), so for every projection ONE TMA tensor copy
//    (cp.async.bulk.tensor.4d, out-of-bounds pixels arrive as zeros = the detector edge for free) brings the D-channel
//    tile of wr the whole brick needs into shared memory, a ring of NST stages deep.  The gather then reads its
//    candidate rays from shared memory at fixed offsets: no global-load latency, no address arithmetic, no bounds
//    predicates (round 1 gathered from global memory: 414 thread-instructions per voxel-projection, a third of the
//    time stalled on the loads, profiles/r01_ncu_c5_v5.md).
//  * Positions inside the tile are small numbers (< 16), so fp32 carries them to ~1e-6 pixel; the tile origin is
//    computed in fp64 by the producer warp, 32 projections at a time (one per lane).
//  * The contraction over (s, c) runs on the 5th-generation tensor cores exactly as before (tcgen05.mma kind::tf32,
//    M = 128, N = ldk, K = 8, 3xTF32 split, windowed accumulation against the truncating fp32 adder), but the A
//    operand (the gathered values, hi and lo parts) is written straight to TENSOR MEMORY by its row's thread
//    (tcgen05.st) and read from there by the MMA: it never touches shared memory.  The B operand (w_s B_s, split and
//    laid out once per call by bop_prep_kernel) arrives with the tile through a second bulk copy.
//  * Warp roles: 0-3 gather, 4 TMA producer, 5 MMA issuer; full/empty mbarriers per stage, no block-wide barrier in
//    the projection loop.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

#include <atomic>
#include <mutex>
#include <string>

#include "mm_internal.h"
#include "mm_ptx.cuh"

using namespace mmptx;

namespace {

// brick of voxels per CTA; thread t = 32 warp + lane holds voxel (dx, dy, dz) = (lane bit 2 | warp bit 1 << 1,
// lane bit 1 | warp bit 0 << 1, lane bit 0 | lane bits 3-4 << 1): the eight lanes of a quarter-warp (one shared-memory
// access phase) form a 2 x 2 x 2 cube, whose shadow on the detector spans at most 3 x 3 pixels — pixel indices that the
// swizzled tile keeps in different banks
constexpr int BX = 4, BY = 4, BZ = 8;
constexpr int NTHREADS = 192;
constexpr int NST = 4;                             // tile ring depth
constexpr int WIN_MMAS = 48;                       // MMAs per accumulation window (see drain_window)
constexpr float MAGIC = 12582912.f;                // 1.5 * 2^23: x + MAGIC has round-to-nearest(x) in its low mantissa bits
constexpr uint32_t MAGIC_BITS = 0x4B400000u;

struct BrickArgs {
    const MMProj *tab;
    const float *bop;         // [P][hi, lo][D/4][NPAD][4]: split operand tiles of w_s B_s (bop_prep_kernel)
    float *out;               // [X][Y][Z][ldk]
    int ldk, X, Y, Z, P;
    int x_begin, x_end;       // planes of x written by this launch
    int nby, nbz;             // bricks along y and z
    int tj, tk;               // tile box in pixels
    int tile_stride;          // bytes between tile stages (multiple of 128)
    int bilinear;
};

// Per-stage constants written by the producer for the gather threads, four float4 per stage:
//   [0] Jx0, Jx1, Jx2, base_lj     local detector position: lj = base_lj + dx Jx0 + dy Jx1 + dz Jx2
//   [1] Kx0, Kx1, Kx2, base_lk
//   [2] mju, mku, mjv, mkv         in-slab displacement of a ray offset (dj, dk): du = mju dj + mku dk, dv = mjv dj + mkv dk
//   [3] code (as int bits): 2 (NJ - 2) + (NK - 2), NJ, NK = candidate window widths

template <int D, int NPAD>
struct Cfg {
    static constexpr int BOP_BYTES = 2 * NPAD * D * 4;
    static constexpr int ACOLS = 2 * D;                                   // hi | lo columns of one A stage
    static constexpr int USED = 2 * NPAD + 2 * ACOLS;                     // acc | running sum | A ring (2 stages)
    static constexpr int TCOLS = USED <= 32 ? 32 : USED <= 64 ? 64 : USED <= 128 ? 128 : USED <= 256 ? 256 : 512;
    static constexpr int WIN = WIN_MMAS / (3 * (D / 8));                  // projections per accumulation window
    static constexpr int MINB = 512 / TCOLS < 4 ? 512 / TCOLS : 4;
    static_assert(USED <= 512, "tensor memory");
};

// two adjacent floats as one 64-bit register pair: sm_100 has packed fp32 arithmetic (fma.rn.f32x2 -> FFMA2), which
// halves the issue slots of the gather's multiply-adds
typedef unsigned long long f32x2;
__device__ __forceinline__ void lds_2x2(uint32_t addr, f32x2 &a, f32x2 &b)
{
    asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "r"(addr));
}
__device__ __forceinline__ f32x2 pack2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ void fma2(f32x2 &acc, f32x2 w, f32x2 v) { asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(w), "l"(v)); }

// t[c] += w * tile[addr + 4 c] (t as D/2 packed pairs).  About half of the candidates of a window have zero weight;
// with SKIP their lanes read a block of zeros instead (one address for all of them: a broadcast).
//
// The tile sits in shared memory with TMA's swizzle of one pixel's width (32 bytes for D = 8, 64 for D = 16): the low
// bit(s) of the 16-byte chunk index (address bits 4..) are XORed with the low bit(s) of the 128-byte row index (bits
// 7..).  Unswizzled, the eight lanes of a quarter-warp could use only four of the eight 16-byte bank groups (all lanes
// read the same chunk of their pixel): every tile read was a 2-way conflict (ncu, round-2 v1: 91 wavefronts per warp
// and projection against 47 ideal, L1 data pipe at 87 %).  Swizzled, lanes whose pixel indices differ mod 8 never collide.
template <int D, bool SKIP>
__device__ __forceinline__ void acc_candidate(float w, uint32_t addr, uint32_t zeros, f32x2 (&t)[D / 2])
{
    static_assert(D == 8 || D == 16, "D");
    addr ^= (addr >> 3) & (D == 8 ? 0x10u : 0x30u);                  // a pixel never straddles a 128-byte row
    if (SKIP) addr = w > 0.f ? addr : zeros;
    const f32x2 w2 = pack2(w, w);
#pragma unroll
    for (int c = 0; c < D; c += 4) {
        // chunk c/4 of the pixel: the pixel is aligned to its size, so adding 4c bytes to the unswizzled address only
        // sets low chunk-index bits that are zero there — the same as XORing them into the swizzled address
        f32x2 a, b;
        lds_2x2(addr ^ (uint32_t)(4 * c), a, b);
        fma2(t[c / 2], w2, a);
        fma2(t[c / 2 + 1], w2, b);
    }
}

// Gather of one voxel from the staged tile, candidate window NJ x NK rays (2 or 3 wide).  Candidate (r, c) sits at a
// fixed offset from the first one; its in-slab displacement is affine in (r, c), so the weights cost two adds, two
// saturating adds (Lambda(t) = sat(1 - |t|)) and a multiply.  Pixels off the detector hold zeros (TMA), rays outside
// the support have zero weight: no predicate is needed for correctness.
//   3-wide: integers within 1.5 of l are {n-1, n, n+1}, n = round(l);  2-wide: within 1 of l are {floor l, floor l + 1}.
template <int D, int NJ, int NK, bool SKIP>
__device__ __forceinline__ void gather_tile(const float4 cj, const float4 ck, const float4 cm, uint32_t tile, int pitch, uint32_t bias,
                                            uint32_t zeros, float dxf, float dyf, float dzf, f32x2 (&t)[D / 2])
{
    // cj = (Jx0, Jx1, Jx2, base_lj), ck = (Kx0, Kx1, Kx2, base_lk), cm = (mju, mku, mjv, mkv)
    const float lj = fmaf(dxf, cj.x, fmaf(dyf, cj.y, fmaf(dzf, cj.z, cj.w)));
    const float lk = fmaf(dxf, ck.x, fmaf(dyf, ck.y, fmaf(dzf, ck.z, ck.w)));
    const float tj = __fadd_rn(lj, MAGIC), tk = __fadd_rn(lk, MAGIC);
    const float fj = lj - __fadd_rn(tj, -MAGIC), fk = lk - __fadd_rn(tk, -MAGIC);     // l - round(l), in [-0.5, 0.5]
    int nj = __float_as_int(tj), nk = __float_as_int(tk);                            // round(l) + MAGIC_BITS
    float ej, ek;                                                                     // first candidate minus l
    if (NJ == 3) { ej = -1.f - fj; nj -= 1; } else { const bool neg = fj < 0.f; ej = (neg ? -1.f : 0.f) - fj; nj -= neg ? 1 : 0; }
    if (NK == 3) { ek = -1.f - fk; nk -= 1; } else { const bool neg = fk < 0.f; ek = (neg ? -1.f : 0.f) - fk; nk -= neg ? 1 : 0; }
    uint32_t addr = tile + (uint32_t)nj * (uint32_t)pitch + (uint32_t)nk * (uint32_t)(D * 4) - bias;
    float du0 = fmaf(cm.x, ej, cm.y * ek), dv0 = fmaf(cm.z, ej, cm.w * ek);
#pragma unroll
    for (int r = 0; r < NJ; r++) {
        float du = du0, dv = dv0;
#pragma unroll
        for (int q = 0; q < NK; q++) {
            const float w = __saturatef(1.f - fabsf(du)) * __saturatef(1.f - fabsf(dv));
            acc_candidate<D, SKIP>(w, addr + q * (D * 4), zeros, t);
            du += cm.y; dv += cm.w;
        }
        du0 += cm.x; dv0 += cm.z;
        addr += pitch;
    }
}

// SKIP = 1 redirects the reads of zero-weight candidates to a block of zeros.  Measured on config 5 with the cube lane
// mapping and the swizzled tile: 62.5 ms with, 57.1 ms without (the select costs more issue slots than the saved
// wavefronts are worth once the reads are conflict-free); kept as a compile-time switch.
#ifndef MM_BRICK_SKIP
#define MM_BRICK_SKIP 0
#endif

template <int D, int NPAD>
__global__ void __launch_bounds__(NTHREADS, Cfg<D, NPAD>::MINB)
adjoint_brick_kernel(const __grid_constant__ CUtensorMap tmap, const BrickArgs a)
{
    using C = Cfg<D, NPAD>;
    constexpr int WIN = C::WIN;
    constexpr uint32_t IDESC = idesc_tf32(128, NPAD);
    extern __shared__ __align__(1024) unsigned char smem[];
    // [tiles NST x tile_stride][B operands NST x BOP_BYTES][stage constants NST x 64][64 zero bytes][barriers][tmem slot]
    const uint32_t s_tiles = smem_u32(smem);
    const uint32_t s_bop = s_tiles + NST * a.tile_stride;
    unsigned char *tail = smem + NST * a.tile_stride + NST * C::BOP_BYTES;
    float4 *cst = reinterpret_cast<float4 *>(tail);
    float *zero_block = reinterpret_cast<float *>(tail + NST * 64);  // 64-byte aligned block of zeros (see acc_candidate)
    const uint32_t s_bar = smem_u32(tail + NST * 64 + 64);
    const uint32_t full_tile = s_bar, empty_tile = s_bar + 8 * NST, full_a = s_bar + 16 * NST, empty_a = full_a + 16,
                   wbar = full_a + 32, drained = full_a + 40;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tail + NST * 64 + 64 + 16 * NST + 48);
    constexpr bool SKIP = MM_BRICK_SKIP != 0;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int P = a.P;
    // brick of this CTA: z fastest, so neighbouring CTAs share detector tiles in L2
    const int bz = blockIdx.x % a.nbz, by = (blockIdx.x / a.nbz) % a.nby, bx = blockIdx.x / (a.nbz * a.nby);
    const int x0 = a.x_begin + bx * BX, y0 = by * BY, z0 = bz * BZ;

    if (warp == 5) tmem_alloc<C::TCOLS>(smem_u32(tmem_slot));
    if (tid == 0) {
        for (int i = 0; i < NST; i++) { mbar_init(full_tile + 8 * i, 1); mbar_init(empty_tile + 8 * i, 5); }
        mbar_init(full_a, 4); mbar_init(full_a + 8, 4);
        mbar_init(empty_a, 1); mbar_init(empty_a + 8, 1);
        mbar_init(wbar, 1); mbar_init(drained, 4);
        mbar_fence_init();
    }
    if ((s_tiles & 1023u) != 0) __trap();                            // swizzled TMA destinations need 1024-byte alignment
    if (tid == 128) tma_prefetch_desc(&tmap);
    if (tid < 16) zero_block[tid] = 0.f;
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tm = *tmem_slot;                                  // columns: [0,NPAD) acc | [NPAD,2NPAD) sum | A ring
    const uint32_t tm_a = tm + 2 * NPAD;

    if (warp == 4) {
        // ---------------- producer: tile origin + constants, TMA tile, bulk B operand ----------------
        for (int sb = 0; sb < P; sb += 32) {
            // lane l prepares projection sb + l (all fp64 work of 32 projections in parallel)
            const int s = min(sb + lane, P - 1);
            const MMProj *pg = a.tab + s;
            const double Jx0 = pg->Jx[0], Jx1 = pg->Jx[1], Jx2 = pg->Jx[2], Kx0 = pg->Kx[0], Kx1 = pg->Kx[1], Kx2 = pg->Kx[2];
            const double j0 = fma((double)x0, Jx0, fma((double)y0, Jx1, fma((double)z0, Jx2, pg->Jc)));
            const double k0 = fma((double)x0, Kx0, fma((double)y0, Kx1, fma((double)z0, Kx2, pg->Kc)));
            const double minj = j0 + fmin(0.0, (BX - 1) * Jx0) + fmin(0.0, (BY - 1) * Jx1) + fmin(0.0, (BZ - 1) * Jx2);
            const double mink = k0 + fmin(0.0, (BX - 1) * Kx0) + fmin(0.0, (BY - 1) * Kx1) + fmin(0.0, (BZ - 1) * Kx2);
            // tile origin two pixels below the nearest pixel of the brick's lowest corner: local positions start in
            // [1.5, 2.5], so the first candidate (round(l) - 1) is never negative
            const int jb0 = __double2int_rn(minj) - 2, kb0 = __double2int_rn(mink) - 2;
            const float4 cj = make_float4((float)Jx0, (float)Jx1, (float)Jx2, (float)(j0 - (double)jb0));
            const float4 ck = make_float4((float)Kx0, (float)Kx1, (float)Kx2, (float)(k0 - (double)kb0));
            // bilinear: weights (1-fj | fj)(1-fk | fk) = the 2 x 2 window with M = identity
            const float4 cm = a.bilinear ? make_float4(1.f, 0.f, 0.f, 1.f) : make_float4(pg->mju, pg->mku, pg->mjv, pg->mkv);
            const float4 cc = make_float4(__int_as_float(a.bilinear ? 0 : pg->gcode - 4), 0.f, 0.f, 0.f);
            const int n = min(32, P - sb);
            for (int i = 0; i < n; i++) {
                const int sp = sb + i, st = sp % NST, use = sp / NST;
                if (lane == i) {
                    if (use > 0) mbar_wait(empty_tile + 8 * st, (uint32_t)((use - 1) & 1));
                    cst[4 * st] = cj; cst[4 * st + 1] = ck; cst[4 * st + 2] = cm; cst[4 * st + 3] = cc;
                    const uint32_t bar = full_tile + 8 * st;
                    mbar_arrive_expect_tx(bar, (uint32_t)(a.tj * a.tk * D * 4 + C::BOP_BYTES));
                    tma_load_4d(s_tiles + st * a.tile_stride, &tmap, bar, 0, kb0, jb0, sp);
                    bulk_load(s_bop + st * C::BOP_BYTES, a.bop + (size_t)sp * (C::BOP_BYTES / 4), C::BOP_BYTES, bar);
                }
                __syncwarp();
            }
        }
    } else if (warp == 5) {
        // ---------------- MMA issuer ----------------
        if (lane == 0) {
            for (int s = 0; s < P; s++) {
                const int st = s % NST, sa = s & 1;
                mbar_wait(full_tile + 8 * st, (uint32_t)((s / NST) & 1));          // B operand has landed
                mbar_wait(full_a + 8 * sa, (uint32_t)((s >> 1) & 1));             // all 128 rows of A are in tensor memory
                if (s % WIN == 0 && s > 0) mbar_wait(drained, (uint32_t)((s / WIN - 1) & 1));   // previous window has left acc
                tc_fence_after();
                const uint32_t b_hi = s_bop + st * C::BOP_BYTES, b_lo = b_hi + C::BOP_BYTES / 2;
                const uint32_t a_hi = tm_a + sa * C::ACOLS, a_lo = a_hi + D;
#pragma unroll
                for (int ks = 0; ks < D / 8; ks++) {
                    const uint32_t bo = ks * 2 * (NPAD * 16);
                    const uint64_t dBh = smem_desc(b_hi + bo, NPAD * 16, 128), dBl = smem_desc(b_lo + bo, NPAD * 16, 128);
                    mma_tf32_ts(tm, a_lo + 8 * ks, dBh, IDESC, ((s % WIN) | ks) ? 1u : 0u);       // small terms first
                    mma_tf32_ts(tm, a_hi + 8 * ks, dBl, IDESC, 1u);
                    mma_tf32_ts(tm, a_hi + 8 * ks, dBh, IDESC, 1u);
                }
                tc_commit(empty_a + 8 * sa);
                tc_commit(empty_tile + 8 * st);
                if (s % WIN == WIN - 1 || s == P - 1) tc_commit(wbar);
            }
        }
        __syncwarp();
    } else {
        // ---------------- gather warps ----------------
        const int dz = (lane & 1) | ((lane >> 3) << 1), dy = ((lane >> 1) & 1) | ((warp & 1) << 1), dx = ((lane >> 2) & 1) | ((warp >> 1) << 1);
        const float dxf = (float)dx, dyf = (float)dy, dzf = (float)dz;
        const int pitch = a.tk * D * 4;
        const uint32_t bias = MAGIC_BITS * (uint32_t)pitch + MAGIC_BITS * (uint32_t)(D * 4);
        const uint32_t lane_base = tm + ((uint32_t)(warp * 32) << 16);
        const uint32_t zeros = smem_u32(zero_block);
        // The tensor core adds into its fp32 accumulator with truncation (measured in round 1: -3e-8 relative per
        // accumulation, -1.6e-5 over config 5's 1080 MMAs), so accumulation is cut into windows of WIN_MMAS MMAs; each
        // finished window is added in round-to-nearest fp32 to a running sum kept in tensor memory.  The drain of
        // window w is deferred until this thread has handed over the first projection of window w + 1, so the MMAs of
        // the window's tail are long complete when it looks.
        auto drain_window = [&](int w) {
            mbar_wait(wbar, (uint32_t)(w & 1));
            tc_fence_after();
#pragma unroll
            for (int c0 = 0; c0 < NPAD; c0 += 16) {
                float v[16];
                tmem_ld16(lane_base + c0, v);
                if (w > 0) {
                    float m[16];
                    tmem_ld16(lane_base + NPAD + c0, m);
#pragma unroll
                    for (int i = 0; i < 16; i++) v[i] += m[i];
                }
                uint32_t u[16];
#pragma unroll
                for (int i = 0; i < 16; i++) u[i] = __float_as_uint(v[i]);
                tmem_st16(lane_base + NPAD + c0, u);
            }
            tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(drained);
        };

        for (int s = 0; s < P; s++) {
            const int st = s % NST, sa = s & 1;
            mbar_wait(full_tile + 8 * st, (uint32_t)((s / NST) & 1));
            const float4 cj = cst[4 * st], ck = cst[4 * st + 1], cm = cst[4 * st + 2];
            const int code = __float_as_int(cst[4 * st + 3].x);
            const uint32_t tile = s_tiles + st * a.tile_stride;
            f32x2 t2[D / 2];
#pragma unroll
            for (int i = 0; i < D / 2; i++) t2[i] = 0ull;
            switch (code) {                                           // uniform across the block
                case 0: gather_tile<D, 2, 2, SKIP>(cj, ck, cm, tile, pitch, bias, zeros, dxf, dyf, dzf, t2); break;
                case 1: gather_tile<D, 2, 3, SKIP>(cj, ck, cm, tile, pitch, bias, zeros, dxf, dyf, dzf, t2); break;
                case 2: gather_tile<D, 3, 2, SKIP>(cj, ck, cm, tile, pitch, bias, zeros, dxf, dyf, dzf, t2); break;
                default: gather_tile<D, 3, 3, SKIP>(cj, ck, cm, tile, pitch, bias, zeros, dxf, dyf, dzf, t2); break;
            }
            float t[D];
#pragma unroll
            for (int i = 0; i < D / 2; i++) unpack2(t2[i], t[2 * i], t[2 * i + 1]);
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_tile + 8 * st);          // this warp is done with the tile
            if (s >= 2) { mbar_wait(empty_a + 8 * sa, (uint32_t)(((s >> 1) - 1) & 1)); tc_fence_after(); }
            const uint32_t arow = lane_base + (uint32_t)(2 * NPAD + sa * C::ACOLS);
            if constexpr (D == 8) {
                uint32_t u[16];
#pragma unroll
                for (int i = 0; i < 8; i++) split_tf32(t[i], u[i], u[8 + i]);
                tmem_st16(arow, u);
            } else {
                uint32_t hi[16], lo[16];
#pragma unroll
                for (int i = 0; i < 16; i++) split_tf32(t[i], hi[i], lo[i]);
                tmem_st16(arow, hi);
                tmem_st16(arow + 16, lo);
            }
            tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(full_a + 8 * sa);
            if (s % WIN == 0 && s > 0) drain_window(s / WIN - 1);
        }
        // epilogue: last window + running sum -> grad (thread = voxel)
        const int wl = (P - 1) / WIN;
        mbar_wait(wbar, (uint32_t)(wl & 1));
        tc_fence_after();
        const int x = x0 + dx, y = y0 + dy, z = z0 + dz;
        const bool ok = x < a.x_end && y < a.Y && z < a.Z;
        float *o = a.out + (((long long)x * a.Y + y) * a.Z + z) * a.ldk;
#pragma unroll
        for (int c0 = 0; c0 < NPAD; c0 += 16) {
            float v[16];
            tmem_ld16(lane_base + c0, v);
            if (wl > 0) {
                float m[16];
                tmem_ld16(lane_base + NPAD + c0, m);
#pragma unroll
                for (int i = 0; i < 16; i++) v[i] += m[i];
            }
            if (ok) {
#pragma unroll
                for (int i = 0; i < 16; i += 4)
                    if (c0 + i < a.ldk)                 // ldk % 4 == 0 on this path; rows K..ldk-1 of B are zero
                        *reinterpret_cast<float4 *>(o + c0 + i) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 5) tmem_dealloc<C::TCOLS>(tm);
}

// w_s B[s][i][c] -> split hi/lo operand tiles in the K-major no-swizzle layout of the shared-memory descriptor:
// element (n = channel i, k = c) at (k/4) * (NPAD*16) + n*16 + (k%4)*4 bytes; rows K..NPAD-1 are zero.
__global__ void bop_prep_kernel(const float *__restrict__ B, const MMProj *__restrict__ tab, float *__restrict__ bop, int K, int D,
                                int NPAD)
{
    const int s = blockIdx.x;
    const float w = tab[s].w;
    float *hi = bop + (size_t)s * (2 * NPAD * D), *lo = hi + NPAD * D;
    for (int g = threadIdx.x; g < NPAD * (D / 4); g += blockDim.x) {
        const int n = g % NPAD, kg = g / NPAD;
        float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
        if (n < K) {
            b = __ldg(reinterpret_cast<const float4 *>(B + ((size_t)s * K + n) * D + 4 * kg));
            b.x *= w; b.y *= w; b.z *= w; b.w *= w;
        }
        uint32_t h[4], l[4];
        split_tf32(b.x, h[0], l[0]); split_tf32(b.y, h[1], l[1]); split_tf32(b.z, h[2], l[2]); split_tf32(b.w, h[3], l[3]);
        *reinterpret_cast<uint4 *>(hi + kg * (NPAD * 4) + n * 4) = make_uint4(h[0], h[1], h[2], h[3]);
        *reinterpret_cast<uint4 *>(lo + kg * (NPAD * 4) + n * 4) = make_uint4(l[0], l[1], l[2], l[3]);
    }
}

template <int D, int NPAD>
cudaError_t launch_brick(const CUtensorMap &tmap, const BrickArgs &a, cudaStream_t st)
{
    using C = Cfg<D, NPAD>;
    const size_t smem = (size_t)NST * a.tile_stride + (size_t)NST * C::BOP_BYTES + NST * 64 + 64 + 16 * NST + 48 + 16;
    // per launch: the attribute is per device, and this is cheaper than tracking which devices have it
    cudaError_t e = cudaFuncSetAttribute(adjoint_brick_kernel<D, NPAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int nbx = (a.x_end - a.x_begin + BX - 1) / BX;
    const long long grid = (long long)nbx * a.nby * a.nbz;
    if (grid <= 0) return cudaSuccess;
    adjoint_brick_kernel<D, NPAD><<<(unsigned)grid, NTHREADS, smem, st>>>(tmap, a);
    return cudaGetLastError();
}

#include "mm_adjoint_brick_pair.cuh"

int npad_for(int ldk)
{
    return ldk <= 16 ? 16 : ldk <= 32 ? 32 : ldk <= 48 ? 48 : ldk <= 64 ? 64 : ldk <= 96 ? 96 : ldk <= 128 ? 128 : 192;
}

}  // namespace

bool mm_adjoint_brick_supported(const mm_geometry *g, const AdjArgs &a)
{
    const long long plane = (long long)a.Y * a.Z;
    return g->brick_tj > 0 && (a.D == 8 || a.D == 16) && a.ldk % 4 == 0 && a.ldk <= 192 && a.vec_ok &&
           (reinterpret_cast<uintptr_t>(a.B) & 15u) == 0 && (reinterpret_cast<uintptr_t>(a.out) & 15u) == 0 &&
           (reinterpret_cast<uintptr_t>(a.src) & 15u) == 0 && a.vox_begin % plane == 0 && a.vox_end % plane == 0 &&
           (a.vox_begin / plane) % BX == 0 && (long long)a.P * a.J * a.Kd * a.D < (1LL << 40) && mm_tma_available();
}

int mm_adjoint_brick_launch(const mm_geometry *g, const AdjArgs &a, void *stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    const long long plane = (long long)a.Y * a.Z;
    BrickArgs b;
    b.tab = a.tab; b.out = a.out; b.ldk = a.ldk; b.X = a.X; b.Y = a.Y; b.Z = a.Z; b.P = a.P;
    b.x_begin = (int)(a.vox_begin / plane); b.x_end = (int)(a.vox_end / plane);
    if (b.x_end <= b.x_begin) return cudaSuccess;
    b.nby = (a.Y + BY - 1) / BY; b.nbz = (a.Z + BZ - 1) / BZ;
    b.tj = g->brick_tj; b.tk = g->brick_tk;
    b.tile_stride = (b.tj * b.tk * a.D * 4 + 1023) & ~1023;            // swizzled tiles: 1024-byte aligned stages
    b.bilinear = a.bilinear;
    alignas(64) CUtensorMap tmap;
    const unsigned long long n[4] = {(unsigned long long)a.D, (unsigned long long)a.Kd, (unsigned long long)a.J, (unsigned long long)a.P};
    const unsigned box[4] = {(unsigned)a.D, (unsigned)b.tk, (unsigned)b.tj, 1u};
    if (!mm_tma_encode_4d_f32(&tmap, a.src, n, box, a.D * 4)) return cudaErrorInvalidValue;
    const int NP = npad_for(a.ldk);
    float *bop = nullptr;
    cudaError_t e = mm_scratch_alloc((void **)&bop, (size_t)a.P * 2 * NP * a.D * sizeof(float), st);
    if (e != cudaSuccess) return e;
    b.bop = bop;
    bop_prep_kernel<<<a.P, 128, 0, st>>>(a.B, a.tab, bop, a.K, a.D, NP);
    e = cudaGetLastError();
    // D = 8: two projections per pipeline stage (mm_adjoint_brick_pair.cuh: bit-identical, 5 % faster on config 5);
    // MM_DISABLE_BRICK_PAIR keeps the one-projection kernel
    static const bool pair_on = getenv("MM_DISABLE_BRICK_PAIR") == nullptr;
#define MM_BRICK_CASE(DD, NN) if (e == cudaSuccess && a.D == DD && NP == NN) e = (pair_on && DD == 8) ? launch_brick_pair<NN>(tmap, b, st) : launch_brick<DD, NN>(tmap, b, st)
    MM_BRICK_CASE(8, 16); MM_BRICK_CASE(8, 32); MM_BRICK_CASE(8, 48); MM_BRICK_CASE(8, 64);
    MM_BRICK_CASE(8, 96); MM_BRICK_CASE(8, 128); MM_BRICK_CASE(8, 192);
    MM_BRICK_CASE(16, 16); MM_BRICK_CASE(16, 32); MM_BRICK_CASE(16, 48); MM_BRICK_CASE(16, 64);
    MM_BRICK_CASE(16, 96); MM_BRICK_CASE(16, 128); MM_BRICK_CASE(16, 192);
#undef MM_BRICK_CASE
    const cudaError_t e2 = mm_scratch_free(bop, st);
    return e != cudaSuccess ? e : e2;
}

// ================================================================================================
// mm_adjoint_noalloc: the same brick adjoint for callers that may not allocate (include/mm.h)
// ================================================================================================
// The one piece of scratch the brick adjoint needs is the split operand tiles of w_s B_s (bop_prep_kernel's output,
// P x 2 x NPAD x D floats: 1.1 MB on config 5).  Here they live in a file-scope device array instead of the pool:
// every GPU that loads the library holds MM_ADJOINT_NOALLOC_MAX_BYTES until the process exits.  All calls share the
// array; bop_prep_kernel rewrites every element the brick kernel reads (rows K..NPAD-1 as zeros), so nothing carried
// over from an earlier call is ever used — but two calls in flight on the GPU at once (different streams) race on it.
static __device__ __align__(256) float g_bop_static[MM_ADJOINT_NOALLOC_MAX_BYTES / sizeof(float)];

namespace {
// `g_bop_static` in host code names a host-side shadow, not device memory: the device address comes from
// cudaGetSymbolAddress, asked once per device with that device current.
constexpr int MAX_DEVICES = 64;
float *g_bop_static_addr[MAX_DEVICES];          // guarded by the acquire/release pair below
std::atomic<int> g_bop_static_ready[MAX_DEVICES];

cudaError_t static_bop_address(int dev, float **out)
{
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    if (!g_bop_static_ready[dev].load(std::memory_order_acquire)) {
        static std::mutex mu;
        std::lock_guard<std::mutex> lock(mu);
        if (!g_bop_static_ready[dev].load(std::memory_order_relaxed)) {
            int cur = -1;
            cudaError_t e = cudaGetDevice(&cur);
            if (e != cudaSuccess) return e;
            if (cur != dev) return cudaErrorInvalidDevice;          // the caller checked; never look a symbol up on another device
            float *p = nullptr;
            e = cudaGetSymbolAddress((void **)&p, g_bop_static);
            if (e != cudaSuccess) return e;
            if (!p || (reinterpret_cast<uintptr_t>(p) & 255u) != 0) return cudaErrorInvalidSymbol;
            g_bop_static_addr[dev] = p;
            g_bop_static_ready[dev].store(1, std::memory_order_release);
        }
    }
    *out = g_bop_static_addr[dev];
    return cudaSuccess;
}
}  // namespace

extern "C" mm_status mm_adjoint_noalloc(const mm_geometry *g, const float *B, const float *sino, int32_t K, int32_t ldk,
                                        int32_t D, float *vol_out, void *stream)
{
    const char *who = "mm_adjoint_noalloc";
    if (!g) { mm_set_error(std::string(who) + ": NULL geometry"); return MM_ERR_NULL; }
    if (!g->d_table) { mm_set_error(std::string(who) + ": geometry was created without a CUDA device (no CPU fallback)"); return MM_ERR_CUDA; }
    if (!B || !sino || !vol_out) { mm_set_error(std::string(who) + ": NULL buffer"); return MM_ERR_NULL; }
    if (K < 1 || ldk < K || D < 1 || D > MM_MAX_D) { mm_set_error(std::string(who) + ": need 1 <= K <= ldk, 1 <= D <= MM_MAX_D"); return MM_ERR_SHAPE; }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != g->device) {
        cudaGetLastError();
        mm_set_error(std::string(who) + ": the geometry was created on CUDA device " + std::to_string(g->device) +
                     ", the current device is " + std::to_string(dev));
        return MM_ERR_VALUE;
    }
    AdjArgs a;
    a.tab = g->d_table; a.src = sino; a.B = B; a.out = vol_out; a.K = K; a.ldk = ldk; a.D = D;
    a.X = g->shape[0]; a.Y = g->shape[1]; a.Z = g->shape[2]; a.J = g->J; a.Kd = g->Kd; a.P = g->P;
    a.bilinear = 0; a.vox_begin = 0; a.vox_end = (long long)a.X * a.Y * a.Z;
    a.vec_ok = (D % 4 == 0) && (reinterpret_cast<uintptr_t>(sino) & 15u) == 0;
    const int NP = npad_for(ldk);
    const size_t need = (size_t)a.P * 2 * NP * D * sizeof(float);
    if (need > (size_t)MM_ADJOINT_NOALLOC_MAX_BYTES) {
        mm_set_error(std::string(who) + ": P * 2 * npad(ldk) * D * 4 = " + std::to_string(need) + " bytes of operand scratch exceed the static " +
                     std::to_string((size_t)MM_ADJOINT_NOALLOC_MAX_BYTES) + " bytes (MM_ADJOINT_NOALLOC_MAX_BYTES); use mm_adjoint");
        return MM_ERR_UNSUPPORTED;
    }
    if (!mm_adjoint_brick_supported(g, a)) {
        mm_set_error(std::string(who) + ": only the brick kernel's shapes are served without allocation (D = 8 or 16, ldk % 4 == 0, "
                     "ldk <= 192, 16-byte aligned buffers, a geometry whose brick shadow fits a 16 x 17 pixel tile); use mm_adjoint");
        return MM_ERR_UNSUPPORTED;
    }
    float *bop = nullptr;
    cudaError_t e = static_bop_address(dev, &bop);
    if (e != cudaSuccess) {
        cudaGetLastError();
        mm_set_error(std::string(who) + ": cudaGetSymbolAddress(static scratch): " + cudaGetErrorString(e));
        return MM_ERR_CUDA;
    }
    cudaStream_t st = (cudaStream_t)stream;
    BrickArgs b;
    b.tab = a.tab; b.out = a.out; b.ldk = a.ldk; b.X = a.X; b.Y = a.Y; b.Z = a.Z; b.P = a.P;
    b.x_begin = 0; b.x_end = a.X;
    b.nby = (a.Y + BY - 1) / BY; b.nbz = (a.Z + BZ - 1) / BZ;
    b.tj = g->brick_tj; b.tk = g->brick_tk;
    b.tile_stride = (b.tj * b.tk * a.D * 4 + 1023) & ~1023;
    b.bilinear = 0;
    b.bop = bop;
    alignas(64) CUtensorMap tmap;
    const unsigned long long n[4] = {(unsigned long long)a.D, (unsigned long long)a.Kd, (unsigned long long)a.J, (unsigned long long)a.P};
    const unsigned box[4] = {(unsigned)a.D, (unsigned)b.tk, (unsigned)b.tj, 1u};
    if (!mm_tma_encode_4d_f32(&tmap, a.src, n, box, a.D * 4)) { mm_set_error(std::string(who) + ": tensor map encode failed"); return MM_ERR_CUDA; }
    bop_prep_kernel<<<a.P, 128, 0, st>>>(a.B, a.tab, bop, a.K, a.D, NP);      // rewrites every element the brick kernel reads
    e = cudaGetLastError();
    static const bool pair_on = getenv("MM_DISABLE_BRICK_PAIR") == nullptr;     // as mm_adjoint_brick_launch
#define MM_BRICK_CASE(DD, NN) if (e == cudaSuccess && a.D == DD && NP == NN) e = (pair_on && DD == 8) ? launch_brick_pair<NN>(tmap, b, st) : launch_brick<DD, NN>(tmap, b, st)
    MM_BRICK_CASE(8, 16); MM_BRICK_CASE(8, 32); MM_BRICK_CASE(8, 48); MM_BRICK_CASE(8, 64);
    MM_BRICK_CASE(8, 96); MM_BRICK_CASE(8, 128); MM_BRICK_CASE(8, 192);
    MM_BRICK_CASE(16, 16); MM_BRICK_CASE(16, 32); MM_BRICK_CASE(16, 48); MM_BRICK_CASE(16, 64);
    MM_BRICK_CASE(16, 96); MM_BRICK_CASE(16, 128); MM_BRICK_CASE(16, 192);
#undef MM_BRICK_CASE
    if (e != cudaSuccess) {
        cudaGetLastError();
        mm_set_error(std::string(who) + ": " + cudaGetErrorString(e));
        return MM_ERR_CUDA;
    }
    mm_note_launches(2);                                                       // bop_prep_kernel + adjoint_brick_kernel
    return MM_OK;
}
