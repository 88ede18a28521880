// Grouped FP16 x FP16 -> FP32 GEMM on CLUSTERS OF FOUR CTAs (two tcgen05 cta_group::2 pairs) with the A operand
// multicast across the pairs. Used by the persistent engine (persist.cuh); the pair kernel of gemm2sm.cuh stays
// for the round engine.
//
// Why: the pair kernel of gemm2sm.cuh is bound by L2 -> SM bandwidth, not by the tensor pipe (measured on B200:
// ~8.6 TB/s into the SMs at 50-60 % tensor-pipe activity, independent of the SM clock; profiles/). A 256 x 256
// pair tile fetches (256 + 256) x 2 B per k for 2 x 256 x 256 FLOP. Here a cluster computes a 256 x (bn0 + bn1)
// tile, bn <= 256 each: pair p (CTAs 2p, 2p + 1) owns the columns of its half and both pairs share the 256 rows
// of A, which every CTA fetches only half of and multicasts to its sibling in the other pair
// (cp.async.bulk.tensor ... .multicast::cluster): (256 + 512) x 2 B per k for 2 x 256 x 512 FLOP, a quarter less
// L2 -> SM traffic per FLOP, and the sibling's copy crosses the die-to-die link once.
//
// CTA (r, p) = cluster rank 2p + r:  rows [m0 + 128 r, + 128) of A and of the accumulator (its own TMEM),
// columns [n_p + r bn_p / 2, + bn_p / 2) of B. A stage holds 128 x 64 of A (two 64-row boxes; box p is loaded by
// this CTA for itself and for (r, 1 - p), the other box arrives from there) and 64 x (bn_p / 2) of B.
// Barriers: `full` of a stage lives in the pair leader (rank 2p) and counts the bytes landing in both CTAs of
// the pair; `empty` lives in every CTA and needs the tcgen05.commit of BOTH pair leaders (a stage is written
// by the sibling as well); accumulator hand-over (tfull / tempty) is per pair. One scheduler warp (rank 0)
// publishes TileInfo records to all four CTAs.
#pragma once
#include "gemm2sm.cuh"

namespace nolsm {

constexpr int G4_CTAS = 4;

#ifdef NOLSM_TIMING
// probe builds only: cycles spent waiting, summed over CTAs
// 0 mma take, 1 mma tempty, 2 mma full, 3 mma total, 4 epi take, 5 epi tfull, 6 epi work, 7 epi done, 8 prod empty, 9 prod total, 10 prod take
__device__ unsigned long long g4_timing[16];
#define G4_T0() const long long t0_ = clock64()
#define G4_T1(i) tacc_[i] += clock64() - t0_
#define G4_TDECL() long long tacc_[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}
#define G4_TFLUSH(lane0) do { if (lane0) for (int i_ = 0; i_ < 16; ++i_) if (tacc_[i_]) atomicAdd(&g4_timing[i_], (unsigned long long)tacc_[i_]); } while (0)
#else
#define G4_T0()
#define G4_T1(i)
#define G4_TDECL()
#define G4_TFLUSH(lane0)
#endif
// consumers of a TileInfo: per CTA the producer and the epilogue warps, per pair leader the MMA warp
constexpr int G4_TI_CONSUMERS = G4_CTAS * (1 + G2_EPI_WARPS) + 2;

// Column split of an n16-wide GEMM into cluster tiles: pair tiles of 256 columns are taken two at a time; a
// single pair tile left over at the end is cut into two halves (multiples of 16) so that both pairs work.
__host__ __device__ __forceinline__ int g4_ntn(int n16) { return (((n16 + BN - 1) / BN) + 1) >> 1; }
__host__ __device__ __forceinline__ void g4_cols(int n16, int tn, int& n0, int& bn0, int& bn1) {
    const int np = (n16 + BN - 1) / BN;
    n0 = 2 * tn * BN;
    const int w0 = min(BN, n16 - n0);
    if (2 * tn + 1 < np) { bn0 = w0; bn1 = min(BN, n16 - n0 - BN); }
    else { bn0 = (((w0 >> 4) + 1) >> 1) << 4; bn1 = w0 - bn0; }
}

namespace ptx {
// TMA load of one box into the same shared-memory offset of every CTA in `mask`; the bytes are credited to the
// barrier at `bar` (a shared::cluster address with the pair bit cleared: the leader of the executing pair) and to
// the barrier at the same offset in the leader of every destination's pair.
__device__ __forceinline__ void tma_load_2d_pair_mc(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar_cluster, uint16_t mask) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster"
        " [%0], [%1, {%2, %3}], [%4], %5;"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar_cluster), "h"(mask) : "memory");
}
__device__ __forceinline__ void umma_commit_mask(uint32_t bar, uint16_t mask) {
    asm volatile(
        "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
        ::"r"(bar), "h"(mask) : "memory");
}
}  // namespace ptx

// ------------------------------------------------------------------------------------------------
// One-time setup / teardown (all threads of the four CTAs).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t g4_setup(const G2Smem& sm, int warp, int lane) {
    if (warp == G2_WARP_TMA && lane == 0) {
        for (int s = 0; s < G2_STAGES; ++s) { ptx::mbar_init(sm.full(s), 1); ptx::mbar_init(sm.empty(s), 2); }
        for (int a = 0; a < 2; ++a) { ptx::mbar_init(sm.tfull(a), 1); ptx::mbar_init(sm.tempty(a), 2 * G2_EPI_WARPS); }
        for (int q = 0; q < G2_NTI; ++q) { ptx::mbar_init(sm.ti_full(q), 1); ptx::mbar_init(sm.ti_empty(q), G4_TI_CONSUMERS); }
        ptx::mbar_init(sm.want(), 1);
        ptx::fence_mbar_init();
    }
    if (warp == G2_WARP_MMA) ptx::tmem_alloc_pair(sm.tmem_ptr(), 512);
    ptx::tc_fence_before();
    ptx::cluster_sync();
    ptx::tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(sm.tmem_ptr()));
    return tmem_base;
}

// what this CTA's pair does in a tile
struct G4Part {
    int bn, n0;            // columns of the pair (bn == 0: the pair only relays its half of A)
};
__device__ __forceinline__ G4Part g4_part(const TileInfo& ti, uint32_t pair) {
    const int bn0 = ti.bn & 0xFFFF, bn1 = ti.bn >> 16;
    G4Part p;
    p.bn = pair ? bn1 : bn0;
    p.n0 = ti.n0 + (pair ? bn0 : 0);
    return p;
}

// ------------------------------------------------------------------------------------------------
// TMA producer (one warp per CTA; lane 0 issues).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void g4_producer(const G2Smem& sm, const CUtensorMap* maps, uint32_t rank, int lane, int want_lead, int dbg = 0) {
    int stage = 0; uint32_t phase = 0;
    int q = 0; uint32_t tph = 0;
    const uint32_t r = rank & 1u, pair = rank >> 1;
    const uint32_t full0 = ptx::mapa(sm.full(0), rank & ~1u);               // the pair leader's full barriers
    const uint16_t mc_mask = (uint16_t)((1u << r) | (1u << (r + 2)));       // this CTA and its sibling in the other pair
    G4_TDECL();
#ifdef NOLSM_TIMING
    const long long tstart_ = clock64();
#endif
    for (;;) {
        TileInfo ti;
        { G4_T0(); ti = g2_take(sm, q, tph, lane == 0); G4_T1(10); }
        if (++q == G2_NTI) { q = 0; tph ^= 1; }
        if (!ti.valid) break;
        ptx::fence_proxy_async();      // operands may have been written by generic stores of another CTA
        const G4Part pt = g4_part(ti, pair);
        const CUtensorMap* map_a = maps + (size_t)ti.slot * NMAP + ti.a_buf;
        const CUtensorMap* map_b = maps + (size_t)ti.slot * NMAP + ti.b_buf;
        const int nkb = (ti.n16 + BK - 1) / BK;
        const int half = pt.bn >> 1;
        const int nbox = (half + 63) >> 6;
        const uint32_t bytes = 2u * (G2_A_BYTES + nbox * B_BOX_BYTES);     // both CTAs of the pair
        const int arow = ti.m0 + 128 * (int)r + 64 * (int)pair;            // the A box this CTA fetches for both pairs
        const int col0 = pt.n0 + half * (int)r;
        const int kb_want = max(0, nkb - want_lead);
        for (int kb = 0; kb < nkb; ++kb) {
            { G4_T0(); ptx::mbar_wait_cluster(sm.empty(stage), phase ^ 1); G4_T1(8); }
            if (lane == 0) {
                if (kb == kb_want && rank == 0) ptx::mbar_arrive(sm.want());   // the scheduler may claim the next tile now
                const uint32_t fb = full0 + 8u * stage;
#ifdef NOLSM_TIMING
                if (dbg & 2) {                       // probe: no loads, the MMAs run on whatever the stage holds
                    if (r == 0) ptx::mbar_arrive(sm.full(stage));
                } else
#endif
                {
                if (r == 0) ptx::mbar_expect_tx(sm.full(stage), bytes);
                const uint32_t sa = sm.stage_a(stage), sb = sm.stage_b(stage);
                ptx::tma_load_2d_pair_mc(sa + 8192u * pair, map_a, kb * BK, arow, fb, mc_mask);
                for (int b = 0; b < nbox; ++b)
                    ptx::tma_load_2d_pair(sb + b * B_BOX_BYTES, map_b, col0 + b * 64, kb * BK, fb);
                }
            }
            __syncwarp();
            if (++stage == G2_STAGES) { stage = 0; phase ^= 1; }
        }
    }
#ifdef NOLSM_TIMING
    tacc_[9] = clock64() - tstart_;
#endif
    G4_TFLUSH(lane == 0);
}

// ------------------------------------------------------------------------------------------------
// MMA issuer (leader CTA of each pair, one warp; one elected lane issues).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void g4_mma(const G2Smem& sm, uint32_t tmem_base, uint32_t rank, int lane, int dbg = 0) {
    int stage = 0; uint32_t phase = 0;
    int acc = 0; uint32_t acc_phase = 0;
    int q = 0; uint32_t tph = 0;
    const uint32_t pair = rank >> 1;
    const uint16_t pair_mask = (uint16_t)(3u << (2 * pair));
    const uint64_t da0 = make_smem_desc(sm.stage_a(0), 16, 1024);
    const uint64_t db0 = make_smem_desc(sm.stage_b(0), B_BOX_BYTES, 1024);
    G4_TDECL();
#ifdef NOLSM_TIMING
    const long long tstart_ = clock64();
#endif
    for (;;) {
        TileInfo ti;
        { G4_T0(); ti = g2_take(sm, q, tph, lane == 0); G4_T1(0); }
        if (++q == G2_NTI) { q = 0; tph ^= 1; }
        if (!ti.valid) break;
        const G4Part pt = g4_part(ti, pair);
        const int nkb = (ti.n16 + BK - 1) / BK;
        const int ktail = (ti.n16 - (nkb - 1) * BK) >> 4;          // 16-k slices of the last k-block (1..4)
        bool work = pt.bn > 0;
#ifdef NOLSM_TIMING
        const bool real_work = work;
        if (dbg & 1) work = false;                  // probe: no MMAs (loads only)
        const long long tk0_ = clock64();
#endif
        const uint32_t idesc = make_idesc_f16(256, work ? pt.bn : 16);
        if (work) {
            G4_T0();
            ptx::mbar_wait_cluster(sm.tempty(acc), acc_phase ^ 1);
            G4_T1(1);
            ptx::tc_fence_after();
        }
        const uint32_t d_tmem = tmem_base + acc * 256;
        for (int kb = 0; kb < nkb; ++kb) {
            { G4_T0(); ptx::mbar_wait_cluster(sm.full(stage), phase); G4_T1(2); }
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
                if (work) {
                    const uint64_t da = da0 + (uint64_t)(stage * (G2_STAGE_BYTES >> 4));
                    const uint64_t db = db0 + (uint64_t)(stage * (G2_STAGE_BYTES >> 4));
                    if (kb < nkb - 1 || ktail == 4) {
                        ptx::umma_f16_pair_x4(d_tmem, da, db, idesc, kb != 0);
                    } else {
                        for (int k = 0; k < ktail; ++k)
                            ptx::umma_f16_pair(d_tmem, da + 2 * k, db + 128 * k, idesc, (kb | k) != 0);
                    }
                }
                ptx::umma_commit_mask(sm.empty(stage), (uint16_t)0xF);      // the stage is free in all four CTAs (needs both pairs)
                if (work && kb == nkb - 1) ptx::umma_commit_mask(sm.tfull(acc), pair_mask);
            }
            __syncwarp();
            if (++stage == G2_STAGES) { stage = 0; phase ^= 1; }
        }
#ifdef NOLSM_TIMING
        if (real_work && nkb >= 16 && pt.bn == 256) { tacc_[11] += clock64() - tk0_; tacc_[12] += 1; }   // full-width tiles: tempty wait + k-loop
        if ((dbg & 1) && real_work) {               // keep the accumulator protocol alive for the epilogue
            if (ptx::elect_one()) ptx::umma_commit_mask(sm.tfull(acc), pair_mask);
            __syncwarp();
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
#endif
        if (work && ++acc == 2) { acc = 0; acc_phase ^= 1; }
    }
#ifdef NOLSM_TIMING
    tacc_[3] = clock64() - tstart_;
#endif
    G4_TFLUSH(lane == 0);
}

// ------------------------------------------------------------------------------------------------
// Epilogue (warps 0..7 of each CTA): as g2_epilogue, on the pair's columns.
// ------------------------------------------------------------------------------------------------
template <typename Eng, typename Done>
__device__ __forceinline__ void g4_epilogue(const G2Smem& sm, uint32_t tmem_base, const Eng& e, __half* base,
                                            uint32_t rank, int warp, int lane, Done done) {
    int acc = 0; uint32_t acc_phase = 0;
    int q = 0; uint32_t tph = 0;
    const uint32_t r = rank & 1u, pair = rank >> 1;
    const uint32_t tempty0 = ptx::mapa(sm.tempty(0), rank & ~1u);
    const int quarter = warp & 3, chalf = warp >> 2;
    G4_TDECL();
    for (;;) {
        TileInfo ti;
        { G4_T0(); ti = g2_take(sm, q, tph, lane == 0); G4_T1(4); }
        if (++q == G2_NTI) { q = 0; tph ^= 1; }
        if (!ti.valid) break;
        const G4Part pt = g4_part(ti, pair);
        const int n = ti.n, n16 = ti.n16, bn = pt.bn;
        G4_T0();
        if (bn > 0) {
            int ldc;
            __half* C = c_ptr(e, base, ti.slot, ti.c_buf, ldc);
            const bool ident = ti.kind != OP_POW_S && ti.kind != OP_POW_A && ti.kind != OP_DCOLS;
            const int rbase = ti.m0 + 128 * (int)r + quarter * 32;         // first row of this warp
            const int row = rbase + lane;
            const int col0 = pt.n0;
            const float sa = ti.c_out;
            ptx::mbar_wait_sleepy(sm.tfull(acc), acc_phase);
            G4_T1(5);
            ptx::tc_fence_after();
            float rsum = 0.f, vsum = 0.f;
            uint32_t dep = 0;
            for (int c = chalf * 32; c < bn; c += 64) {
                if (col0 + c >= n16 && ti.kind != OP_DCOLS) break;         // warp-uniform
                uint32_t v[32];
                ptx::tmem_ld_32x32(tmem_base + acc * 256 + ((uint32_t)(quarter * 32) << 16) + c, v);
                ptx::tmem_ld_wait();
                dep ^= v[0];
                if (ti.kind == OP_DCOLS) {                             // P[row, 0..31] = acc, FP32 (a6: D columns are formed from FP32)
                    if (c == 0 && row < n16) {
                        float4* prow = reinterpret_cast<float4*>(pcols_ptr(e, ti.slot) + (size_t)row * PCW);
#pragma unroll
                        for (int j = 0; j < PCW; j += 4)
                            prow[j >> 2] = make_float4(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]), __uint_as_float(v[j + 3]));
                    }
                    continue;
                }
                __half* crow = C + (size_t)row * ldc + col0 + c;
                const bool full = (c + 32 <= bn) && (col0 + c + 32 <= n16);
                const bool diag = (col0 + c < rbase + 32) && (col0 + c + 32 > rbase);
                if (full && !diag) {
                    if (row < n16) {
                        float f[32];
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            const float a = __uint_as_float(v[j]);
                            vsum = fmaf(a, a, vsum);
                            f[j] = sa * a;
                        }
#pragma unroll
                        for (int j = 0; j < 32; j += 16) st_half16(crow + j, f + j);
                    }
                } else if (row < n16) {
                    float f[32];
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const int col = col0 + c + j;
                        const float a = __uint_as_float(v[j]);
                        const float delta = (col == row && row < n && ident) ? 1.f : 0.f;
                        const float d = (c + j < bn && col < n16) ? ti.alpha_res * a - delta : 0.f;   // pad rows / columns give exactly 0
                        rsum = fmaf(d, d, rsum);
                        f[j] = ti.c_out * a + ti.beta * delta;
                    }
                    const int cw = min(min(32, bn - c), n16 - (col0 + c));   // 16 or 32 valid columns
#pragma unroll
                    for (int j = 0; j < 32; j += 16)
                        if (j < cw) st_half16(crow + j, f + j);
                }
            }
            ptx::tc_fence_before();
            ptx::fence_proxy_async();      // C is read next through the async proxy (TMA), possibly by another CTA
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_cluster_relaxed(tempty0 + 8u * acc, dep);
            if (ti.want_res) {
                rsum = fmaf(ti.alpha_res * ti.alpha_res, vsum, rsum);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) rsum += __shfl_xor_sync(0xffffffffu, rsum, o);
                if (lane == 0 && rsum != 0.f) atomicAdd(&e.slots[ti.slot].res_acc, rsum);
            }
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(G2_EPI_WARPS * 32) : "memory");   // the CTA's epilogue warps
        G4_T1(6);
        if (warp == 0 && lane == 0) done(ti);
        G4_T1(7);
    }
    G4_TFLUSH(warp == 0 && lane == 0);
}

}  // namespace nolsm
