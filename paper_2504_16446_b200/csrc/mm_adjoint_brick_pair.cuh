// mm_adjoint_brick_pair.cuh — adjoint_brick_kernel with TWO projections per pipeline stage (included by
// mm_adjoint_brick.cu, inside its anonymous namespace; D = 8 only).  Same gather, same MMAs, same windowed accumulation;
// what changes is how often the warps synchronise: one full/empty hand-shake, one A hand-over, one commit per PAIR
// of projections.  ncu on the one-projection kernel (config 5): a third of its instructions and half of its stall
// samples are barrier waits, arrivals, fences and loop control.
//   stage = 2 tiles + 2 operand tiles + 2 constant blocks; NSTP stages.  A operand: one stage of 2 x 2D columns
//   (the same tensor-memory footprint as the two single-projection stages of adjoint_brick_kernel).
constexpr int NSTP = 3;                            // pair stages

template <int D, int NPAD>
__global__ void __launch_bounds__(NTHREADS, Cfg<D, NPAD>::MINB)
adjoint_brick_pair_kernel(const __grid_constant__ CUtensorMap tmap, const BrickArgs a)
{
    using C = Cfg<D, NPAD>;
    constexpr int WIN = C::WIN;
    static_assert(WIN % 2 == 0, "a window of accumulation holds whole pairs");
    constexpr uint32_t IDESC = idesc_tf32(128, NPAD);
    constexpr int NT = 2 * NSTP;                                     // tiles (and operand tiles) in the ring
    extern __shared__ __align__(1024) unsigned char smem[];
    // [tiles NT x tile_stride][B operands NT x BOP_BYTES][constants NT x 64][barriers][tmem slot]
    const uint32_t s_tiles = smem_u32(smem);
    const uint32_t s_bop = s_tiles + NT * a.tile_stride;
    unsigned char *tail = smem + NT * a.tile_stride + NT * C::BOP_BYTES;
    float4 *cst = reinterpret_cast<float4 *>(tail);
    const uint32_t s_bar = smem_u32(tail + NT * 64);
    const uint32_t full_tile = s_bar, empty_tile = s_bar + 8 * NSTP, full_a = s_bar + 16 * NSTP, empty_a = full_a + 8,
                   wbar = full_a + 16, drained = full_a + 24;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tail + NT * 64 + 16 * NSTP + 32);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int P = a.P, NP2 = (P + 1) / 2;                            // pairs
    const int bz = blockIdx.x % a.nbz, by = (blockIdx.x / a.nbz) % a.nby, bx = blockIdx.x / (a.nbz * a.nby);
    const int x0 = a.x_begin + bx * BX, y0 = by * BY, z0 = bz * BZ;

    if (warp == 5) tmem_alloc<C::TCOLS>(smem_u32(tmem_slot));
    if (tid == 0) {
        for (int i = 0; i < NSTP; i++) { mbar_init(full_tile + 8 * i, 1); mbar_init(empty_tile + 8 * i, 5); }
        mbar_init(full_a, 4); mbar_init(empty_a, 1);
        mbar_init(wbar, 1); mbar_init(drained, 4);
        mbar_fence_init();
    }
    if ((s_tiles & 1023u) != 0) __trap();                            // swizzled TMA destinations need 1024-byte alignment
    if (tid == 128) tma_prefetch_desc(&tmap);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tm = *tmem_slot;                                  // columns: [0,NPAD) acc | [NPAD,2NPAD) sum | A: 2 x (hi | lo)
    const uint32_t tm_a = tm + 2 * NPAD;

    if (warp == 4) {
        // ---------------- producer: per pair one wait and one expect_tx; lanes i, i + 1 issue the two projections ----------------
        for (int sb = 0; sb < P; sb += 32) {
            const int s = min(sb + lane, P - 1);
            const MMProj *pg = a.tab + s;
            const double Jx0 = pg->Jx[0], Jx1 = pg->Jx[1], Jx2 = pg->Jx[2], Kx0 = pg->Kx[0], Kx1 = pg->Kx[1], Kx2 = pg->Kx[2];
            const double j0 = fma((double)x0, Jx0, fma((double)y0, Jx1, fma((double)z0, Jx2, pg->Jc)));
            const double k0 = fma((double)x0, Kx0, fma((double)y0, Kx1, fma((double)z0, Kx2, pg->Kc)));
            const double minj = j0 + fmin(0.0, (BX - 1) * Jx0) + fmin(0.0, (BY - 1) * Jx1) + fmin(0.0, (BZ - 1) * Jx2);
            const double mink = k0 + fmin(0.0, (BX - 1) * Kx0) + fmin(0.0, (BY - 1) * Kx1) + fmin(0.0, (BZ - 1) * Kx2);
            const int jb0 = __double2int_rn(minj) - 2, kb0 = __double2int_rn(mink) - 2;
            const float4 cj = make_float4((float)Jx0, (float)Jx1, (float)Jx2, (float)(j0 - (double)jb0));
            const float4 ck = make_float4((float)Kx0, (float)Kx1, (float)Kx2, (float)(k0 - (double)kb0));
            const float4 cm = a.bilinear ? make_float4(1.f, 0.f, 0.f, 1.f) : make_float4(pg->mju, pg->mku, pg->mjv, pg->mkv);
            const float4 cc = make_float4(__int_as_float(a.bilinear ? 0 : pg->gcode - 4), 0.f, 0.f, 0.f);
            const int n = min(32, P - sb);
            for (int i = 0; i < n; i += 2) {
                const int pr = (sb + i) >> 1, stp = pr % NSTP, use = pr / NSTP;
                const int nv = min(2, n - i);                                   // projections in this pair
                const uint32_t bar = full_tile + 8 * stp;
                const bool mine = lane >= i && lane < i + nv;
                const int tix = 2 * stp + (lane - i);
                if (lane == i && use > 0) mbar_wait(empty_tile + 8 * stp, (uint32_t)((use - 1) & 1));
                __syncwarp();
                if (mine) { cst[4 * tix] = cj; cst[4 * tix + 1] = ck; cst[4 * tix + 2] = cm; cst[4 * tix + 3] = cc; }
                __syncwarp();                                                       // both constant blocks are written ...
                if (lane == i) mbar_arrive_expect_tx(bar, (uint32_t)(nv * (a.tj * a.tk * D * 4 + C::BOP_BYTES)));   // ... before the release
                __syncwarp();
                if (mine) {
                    const int sp = sb + lane;
                    tma_load_4d(s_tiles + tix * a.tile_stride, &tmap, bar, 0, kb0, jb0, sp);
                    bulk_load(s_bop + tix * C::BOP_BYTES, a.bop + (size_t)sp * (C::BOP_BYTES / 4), C::BOP_BYTES, bar);
                }
            }
        }
    } else if (warp == 5) {
        // ---------------- MMA issuer ----------------
        if (lane == 0) {
            for (int pr = 0; pr < NP2; pr++) {
                const int stp = pr % NSTP, s0 = 2 * pr, nv = min(2, P - s0);
                mbar_wait(full_tile + 8 * stp, (uint32_t)((pr / NSTP) & 1));       // both B operands have landed
                mbar_wait(full_a, (uint32_t)(pr & 1));                             // all 128 rows of both A operands are in tensor memory
                if (s0 % WIN == 0 && s0 > 0) mbar_wait(drained, (uint32_t)((s0 / WIN - 1) & 1));   // previous window has left acc
                tc_fence_after();
                for (int e = 0; e < nv; e++) {
                    const int s = s0 + e, tix = 2 * stp + e;
                    const uint32_t b_hi = s_bop + tix * C::BOP_BYTES, b_lo = b_hi + C::BOP_BYTES / 2;
                    const uint32_t a_hi = tm_a + e * C::ACOLS, a_lo = a_hi + D;
#pragma unroll
                    for (int ks = 0; ks < D / 8; ks++) {
                        const uint32_t bo = ks * 2 * (NPAD * 16);
                        const uint64_t dBh = smem_desc(b_hi + bo, NPAD * 16, 128), dBl = smem_desc(b_lo + bo, NPAD * 16, 128);
                        mma_tf32_ts(tm, a_lo + 8 * ks, dBh, IDESC, ((s % WIN) | ks) ? 1u : 0u);       // small terms first
                        mma_tf32_ts(tm, a_hi + 8 * ks, dBl, IDESC, 1u);
                        mma_tf32_ts(tm, a_hi + 8 * ks, dBh, IDESC, 1u);
                    }
                }
                tc_commit(empty_a);
                tc_commit(empty_tile + 8 * stp);
                const int sl = s0 + nv - 1;
                if (sl % WIN == WIN - 1 || sl == P - 1) tc_commit(wbar);
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
        // windows of WIN projections against the truncating fp32 adder of the tensor core, as in adjoint_brick_kernel
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

        for (int pr = 0; pr < NP2; pr++) {
            const int stp = pr % NSTP, s0 = 2 * pr, nv = min(2, P - s0);
            mbar_wait(full_tile + 8 * stp, (uint32_t)((pr / NSTP) & 1));
            f32x2 t2[2][D / 2];
#pragma unroll
            for (int e = 0; e < 2; e++) {
#pragma unroll
                for (int i = 0; i < D / 2; i++) t2[e][i] = 0ull;
                if (e < nv) {
                    const int tix = 2 * stp + e;
                    const float4 cj = cst[4 * tix], ck = cst[4 * tix + 1], cm = cst[4 * tix + 2];
                    const int code = __float_as_int(cst[4 * tix + 3].x);
                    const uint32_t tile = s_tiles + tix * a.tile_stride;
                    switch (code) {                                   // uniform across the block
                        case 0: gather_tile<D, 2, 2, false>(cj, ck, cm, tile, pitch, bias, 0u, dxf, dyf, dzf, t2[e]); break;
                        case 1: gather_tile<D, 2, 3, false>(cj, ck, cm, tile, pitch, bias, 0u, dxf, dyf, dzf, t2[e]); break;
                        case 2: gather_tile<D, 3, 2, false>(cj, ck, cm, tile, pitch, bias, 0u, dxf, dyf, dzf, t2[e]); break;
                        default: gather_tile<D, 3, 3, false>(cj, ck, cm, tile, pitch, bias, 0u, dxf, dyf, dzf, t2[e]); break;
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_tile + 8 * stp);         // this warp is done with both tiles
            if (pr >= 1) { mbar_wait(empty_a, (uint32_t)((pr - 1) & 1)); tc_fence_after(); }
            static_assert(D == 8, "pair kernel: D = 8");
#pragma unroll
            for (int e = 0; e < 2; e++) {
                float t[D];
#pragma unroll
                for (int i = 0; i < D / 2; i++) unpack2(t2[e][i], t[2 * i], t[2 * i + 1]);
                uint32_t u[16];
#pragma unroll
                for (int i = 0; i < 8; i++) split_tf32(t[i], u[i], u[8 + i]);
                tmem_st16(lane_base + (uint32_t)(2 * NPAD + e * C::ACOLS), u);
            }
            tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(full_a);
            if (s0 % WIN == 0 && s0 > 0) drain_window(s0 / WIN - 1);
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
                    if (c0 + i < a.ldk)
                        *reinterpret_cast<float4 *>(o + c0 + i) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 5) tmem_dealloc<C::TCOLS>(tm);
}

template <int NPAD>
cudaError_t launch_brick_pair(const CUtensorMap &tmap, const BrickArgs &a, cudaStream_t st)
{
    using C = Cfg<8, NPAD>;
    const size_t smem = (size_t)2 * NSTP * (a.tile_stride + C::BOP_BYTES + 64) + 16 * NSTP + 32 + 16;
    cudaError_t e = cudaFuncSetAttribute(adjoint_brick_pair_kernel<8, NPAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int nbx = (a.x_end - a.x_begin + BX - 1) / BX;
    const long long grid = (long long)nbx * a.nby * a.nbz;
    if (grid <= 0) return cudaSuccess;
    adjoint_brick_pair_kernel<8, NPAD><<<(unsigned)grid, NTHREADS, smem, st>>>(tmap, a);
    return cudaGetLastError();
}
