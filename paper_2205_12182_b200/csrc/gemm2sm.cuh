// Grouped, variable-size FP16 x FP16 -> FP32 GEMM for sm_100a on CTA PAIRS (tcgen05 cta_group::2).
//
// This is the GEMM "C = alpha A B + beta C" the paper counts as 2n^3 FLOP inside the
// matrix iterations (Eq. 6; Schulz inverse, ref [14] PAPER.md:L217).
//
// Two CTAs of a cluster (one TPC) compute one 256 x bn tile (bn <= 256, multiple of 16): CTA r owns
// rows [m0 + 128 r, m0 + 128 r + 128) of A and of the accumulator (its own TMEM) and stages columns
// [n0 + r bn/2, n0 + (r+1) bn/2) of B; the leader CTA issues one tcgen05.mma (M = 256) per 16 k that
// reads both CTAs' shared memory, so every byte of B is fetched from L2 once per pair instead of once
// per CTA (L2 -> SM bytes per FLOP drop by a third against 128 x bn single-CTA tiles).
//
// All matrices are row-major: A is a K-major operand, B an MN-major operand (X * X needs no
// transposed copy of X). TMA boxes are 64 x 64 FP16 with the 128-byte swizzle.
//
// Warp roles per CTA: warps 0-7 epilogue (TMEM lane quarter = warp & 3; the two warps of a quarter take
// alternate 32-column chunks), warp 8 tile scheduler (leader CTA only), warp 9 TMA producer, warp 10
// TMEM allocator + MMA issuer (leader only). The scheduler
// publishes TileInfo records into a small shared-memory ring in BOTH CTAs; every other role consumes
// them in order. The tiles come from the device work queue of the persistent engine (persist.cuh).
#pragma once
#include "gemm_umma.cuh"

namespace nolsm {

// The TMA ring: 4 stages of 32 KB (measured: 3, 4 and 5 stages run at the same speed - the ring is not what bounds the
// k-loop); the fifth 32 KB hold the epilogue's staging boxes for TMA stores of C.
#ifndef G2_STAGES_N
#define G2_STAGES_N 4
#endif
constexpr int G2_STAGES = G2_STAGES_N;
constexpr int G2_CBOX_BYTES = 64 * 64 * 2;            // one 64 x 64 FP16 box of C, 128-byte swizzle (the TMA map's box)
constexpr int G2_CSTAGE_BYTES = 4 * G2_CBOX_BYTES;    // two row groups (64 rows each) x two buffers
constexpr int G2_A_BYTES = 128 * BK * 2;              // 16 KB: this CTA's 128 rows x 64 k
constexpr int G2_B_BYTES = 2 * B_BOX_BYTES;           // 16 KB: 64 k x (up to 128) columns
constexpr int G2_STAGE_BYTES = G2_A_BYTES + G2_B_BYTES;
constexpr int G2_NTI = 4;                             // tile-info ring depth (8 was measured on cfg1 with 1-3 claim credits: 3-10 % slower)
#ifndef G2_WANT_LEAD
#define G2_WANT_LEAD 14                               // k-blocks before the end of its tile at which the producer asks for the next one
#endif
constexpr int G2_EPI_WARPS = 8;                       // warp w: TMEM lane quarter w & 3, column chunks of parity w >> 2
constexpr int G2_WARP_SCHED = 8, G2_WARP_TMA = 9, G2_WARP_MMA = 10;
constexpr int G2_CTRL_THREADS = 11 * 32;              // warps 0..10
// consumers of a TileInfo: leader = producer + MMA + epilogue warps, peer = producer + finisher + epilogue warps
constexpr int G2_TI_CONSUMERS = 2 * (1 + G2_EPI_WARPS) + 2;     // + the finisher warp of the peer CTA

// flags of TileInfo::valid
constexpr int TI_VALID = 1;           // 0 = no more tiles
constexpr int TI_HALF = 2;            // half-height tile (rows m0 .. m0+127, one M = 128 MMA per 16 k: 64 rows per CTA; TMEM lanes
                                      // 0-63 hold columns [0, bn/2), lanes 64-127 columns [bn/2, bn))
constexpr int TI_MIRROR = 4;          // off-diagonal tile of a symmetric product: C^T goes to the block below the diagonal too
constexpr int TI_PLAIN = 8;           // C = c_out acc without identity term; residual = || alpha_res acc ||_F^2 (power iteration, D columns)
constexpr int TI_F32OUT = 16;         // the first PCW accumulator columns go to the slot's FP32 block instead of C (D columns)
constexpr int TI_TRANS = 64;          // tile of the ragged last row block computed transposed: C^T[n0.., m0..] = B^T A_bottom^T, so the
                                      // MMA's M = 256 runs over full columns of C and its N = bn over the r < 256 rows that are left
constexpr int TI_SYMDIAG = 32;        // diagonal tile of a symmetric product: only its upper triangle is stored, and mirrored

struct __align__(16) TileInfo {      // 64 bytes
    int valid;                        // TI_* flags
    int slot, m0, n0;                 // pair tile origin (rows m0 .. m0+255, columns n0 .. n0+bn-1)
    int n, n16, bn, nreports;         // nreports = CTA reports that complete the slot's GEMM
    int a_buf, b_buf, c_buf, want_res;
    float c_out, alpha_res, beta;      // C = c_out * acc + beta * I ; residual || alpha_res * acc - I ||_F^2
    int kind;
};

struct G2Smem {                       // byte offsets from the 1024-aligned base of the CTA's dynamic smem
    uint32_t base;
    __device__ uint32_t stage_a(int s) const { return base + s * G2_STAGE_BYTES; }
    __device__ uint32_t stage_b(int s) const { return base + s * G2_STAGE_BYTES + G2_A_BYTES; }
    __device__ uint32_t stage_c(int group, int buf) const { return base + G2_STAGES * G2_STAGE_BYTES + (group * 2 + buf) * G2_CBOX_BYTES; }
    __device__ uint32_t bars() const { return base + G2_STAGES * G2_STAGE_BYTES + G2_CSTAGE_BYTES; }
    __device__ uint32_t full(int s) const { return bars() + 8u * s; }
    __device__ uint32_t empty(int s) const { return bars() + 8u * (G2_STAGES + s); }
    __device__ uint32_t tfull(int a) const { return bars() + 8u * (2 * G2_STAGES + a); }
    __device__ uint32_t tempty(int a) const { return bars() + 8u * (2 * G2_STAGES + 2 + a); }
    __device__ uint32_t ti_full(int q) const { return bars() + 8u * (2 * G2_STAGES + 4 + q); }
    __device__ uint32_t ti_empty(int q) const { return bars() + 8u * (2 * G2_STAGES + 4 + G2_NTI + q); }
    __device__ uint32_t tmem_ptr() const { return bars() + 8u * (2 * G2_STAGES + 4 + 2 * G2_NTI); }
    // a counter, not a barrier: the tiles whose loads the leader's producer has issued up to the claim point (kb_want)
    __device__ uint32_t want() const { return bars() + 8u * (2 * G2_STAGES + 4 + 2 * G2_NTI) + 8u; }
    // "every store of tile record q is in global memory": one arrival per epilogue warp of both CTAs, in the PEER CTA's
    // shared memory, where the finisher warp waits for it
    __device__ uint32_t cdone(int q) const { return bars() + 8u * (2 * G2_STAGES + 4 + 2 * G2_NTI) + 16u + 8u * q; }
    __device__ uint32_t tinfo(int q) const { return bars() + 512u + 64u * q; }
};
constexpr int G2_SMEM_BYTES = G2_STAGES * G2_STAGE_BYTES + G2_CSTAGE_BYTES + 512 + 64 * G2_NTI + 1024 /*align*/;
static_assert(8 * (2 * G2_STAGES + 4 + 3 * G2_NTI) + 16 <= 512, "barrier area");

namespace ptx {

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t mapa(uint32_t saddr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ void cluster_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// Arrive without memory ordering, for barriers that only hand back a resource whose reads are already
// complete: `dep` is a value loaded from that resource, listed as an operand so the load has retired.
__device__ __forceinline__ void mbar_arrive_cluster_relaxed(uint32_t cluster_addr, uint32_t dep) {
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr), "r"(dep) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait_cluster(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}\n"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// The waits below return false on a stall (watchdog, gemm_umma.cuh).
__device__ __forceinline__ bool mbar_try_wait_cluster_hint(uint32_t bar, uint32_t parity, uint32_t ns) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}\n"
        : "=r"(ok) : "r"(bar), "r"(parity), "r"(ns) : "memory");
    return ok != 0;
}
__device__ __noinline__ bool mbar_wait_cluster_slow(uint32_t bar, uint32_t parity, volatile int* abort_flag, uint32_t ns, uint32_t rounds) {
    unsigned long long t0 = 0;
    for (uint32_t spins = 1;; ++spins) {
        if (mbar_try_wait_cluster_hint(bar, parity, ns)) return true;
        if ((spins & 1023u) == 0 && stalled(t0, abort_flag)) { if (--rounds == 0) return false; t0 = 0; }
    }
}
__device__ __noinline__ bool mbar_wait_cluster_sleep(uint32_t bar, uint32_t parity, volatile int* abort_flag, uint32_t ns, uint32_t rounds) {
    unsigned long long t0 = 0;
    for (uint32_t spins = 1;; ++spins) {
        if (mbar_try_wait_cluster(bar, parity)) return true;
        __nanosleep(ns);
        if ((spins & 4095u) == 0 && stalled(t0, abort_flag)) { if (--rounds == 0) return false; t0 = 0; }
    }
}
__device__ __forceinline__ bool mbar_wait_cluster(uint32_t bar, uint32_t parity, volatile int* abort_flag) {
#pragma unroll 1
    for (int i = 0; i < 4096; ++i)
        if (mbar_try_wait_cluster(bar, parity)) return true;
    return mbar_wait_cluster_sleep(bar, parity, abort_flag, 64u, 1u);
}
// Wait that may legitimately last long (a role of the persistent engine with no work). The scheduler ends such a wait
// with a record that says "no more tiles"; the watchdog only covers a scheduler that is itself stuck, so its limit is
// ten times the usual one.
__device__ __forceinline__ bool mbar_wait_cluster_patient(uint32_t bar, uint32_t parity, volatile int* abort_flag) {
    if (mbar_try_wait_cluster(bar, parity)) return true;
    return mbar_wait_cluster_slow(bar, parity, abort_flag, 4000u, 10u);
}
__device__ __forceinline__ bool mbar_wait_patient(uint32_t bar, uint32_t parity, volatile int* abort_flag) {
    if (mbar_try_wait(bar, parity)) return true;
    return mbar_wait_slow(bar, parity, abort_flag, 4000u, 10u);
}
// Wait of the eight epilogue warps for the accumulator of the tile being multiplied: microseconds long and not on the
// critical path (two accumulators): suspended try_waits (no polling loop).
__device__ __forceinline__ bool mbar_wait_sleepy(uint32_t bar, uint32_t parity, volatile int* abort_flag) {
    if (mbar_try_wait(bar, parity)) return true;
    return mbar_wait_slow(bar, parity, abort_flag, 4000u, 1u);
}
__device__ __forceinline__ void st_cluster_u32(uint32_t cluster_addr, uint32_t v) {
    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(cluster_addr), "r"(v) : "memory");
}
// Asynchronous store of one word into the shared memory of a CTA of the cluster; its 4 bytes are credited to the
// transaction count of an mbarrier of that CTA. A thread that sees the barrier's phase complete (plain CTA-scope wait)
// sees the word: no cluster-scope acquire, hence no L1 invalidation (CCTL.IVALL) on the consumer's side.
__device__ __forceinline__ void st_async_u32(uint32_t cluster_addr, uint32_t v, uint32_t mbar_cluster_addr) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];"
                 ::"r"(cluster_addr), "r"(v), "r"(mbar_cluster_addr) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx_cluster(uint32_t mbar_cluster_addr, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.release.cluster.shared::cluster.b64 _, [%0], %1;" ::"r"(mbar_cluster_addr), "r"(bytes) : "memory");
}
__device__ __forceinline__ uint32_t ld_shared_volatile_u32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void st_shared_volatile_u32(uint32_t addr, uint32_t v) {
    asm volatile("st.volatile.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
// TMA load whose completion bytes are credited to an mbarrier of either CTA of the pair.
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar_cluster, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%2, %3}], [%4], %5;"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar_cluster), "l"(policy) : "memory");
}
// L2 eviction-priority policy for the bulk copies: 1 evict_first, 2 evict_last, else evict_normal.
// The engine loads every operand with evict_first and stores every GEMM result with evict_last: a result must survive in
// L2 until the next GEMM of its chain reads it, some tens of microseconds and several hundred MB of operand traffic later;
// with equal priorities the operand traffic pushes it out to HBM first (measured on cfg2: +5 %, profiles/r02_persist.md).
__device__ __forceinline__ uint64_t l2_policy(int kind) {
    uint64_t p;
    if (kind == 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    else if (kind == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void tmem_alloc_pair(uint32_t smem_dst, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void umma_f16_pair(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}\n"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// arrives (once the MMAs issued so far have completed) on the barrier at the same offset in both CTAs
__device__ __forceinline__ void umma_commit_pair(uint32_t bar) {
    asm volatile(
        "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
        ::"r"(bar), "h"((uint16_t)3) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
// TMA store of one box from shared memory (bulk async-group completion)
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, int c0, int c1, uint32_t src, uint64_t policy) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group.L2::cache_hint [%0, {%1, %2}], [%3], %4;"
                 ::"l"(map), "r"(c0), "r"(c1), "r"(src), "l"(policy) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// 32 halves (16 packed pairs) of one row into a staging box: chunks (16 B) j0 .. j0 + 3 of box row r, 128-byte swizzle
// (chunk ^ (r & 7))
__device__ __forceinline__ void st_box_row(uint32_t box, int r, int j0, const uint32_t* hp) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const uint32_t a = box + (uint32_t)r * 128u + (uint32_t)(((j0 + q) ^ (r & 7)) << 4);
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(hp[4 * q]), "r"(hp[4 * q + 1]), "r"(hp[4 * q + 2]), "r"(hp[4 * q + 3]) : "memory");
    }
}

// The same 32 halves written TRANSPOSED: element j of box row r, column c0 + j goes to box row c0 + j, column r. The lanes
// of a warp are 32 consecutive r: under the swizzle they hit 4 distinct 16-byte chunks of one 128-byte row, 2 lanes per
// bank word: no bank conflict.
__device__ __forceinline__ void st_box_col(uint32_t box, int r, int c0, const uint32_t* hp) {
    const uint32_t rlo = (uint32_t)(r & 7) << 1, rhi = (uint32_t)(r >> 3);
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        const int cc = c0 + j;
        const uint32_t a = box + (uint32_t)cc * 128u + (((rhi ^ (uint32_t)(cc & 7)) << 4) | rlo);
        const unsigned short v = (unsigned short)((j & 1) ? (hp[j >> 1] >> 16) : (hp[j >> 1] & 0xFFFFu));
        asm volatile("st.shared.b16 [%0], %1;" ::"r"(a), "h"(v) : "memory");
    }
}
// Diagonal box of a symmetric product (box rows and box columns are the same index range): the upper triangle of the
// box, element (r, c0 + j) with c0 + j >= r, goes to its own place and to the transposed place.
__device__ __forceinline__ void st_box_sym(uint32_t box, int r, int c0, const uint32_t* hp) {
    const uint32_t rlo = (uint32_t)(r & 7) << 1, rhi = (uint32_t)(r >> 3);
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        const int cc = c0 + j;
        if (cc >= r) {
            const unsigned short v = (unsigned short)((j & 1) ? (hp[j >> 1] >> 16) : (hp[j >> 1] & 0xFFFFu));
            const uint32_t an = box + (uint32_t)r * 128u + (((((uint32_t)cc >> 3) ^ (uint32_t)(r & 7)) << 4) | ((uint32_t)(cc & 7) << 1));
            asm volatile("st.shared.b16 [%0], %1;" ::"r"(an), "h"(v) : "memory");
            if (cc > r) {
                const uint32_t at = box + (uint32_t)cc * 128u + (((rhi ^ (uint32_t)(cc & 7)) << 4) | rlo);
                asm volatile("st.shared.b16 [%0], %1;" ::"r"(at), "h"(v) : "memory");
            }
        }
    }
}

}  // namespace ptx

// ------------------------------------------------------------------------------------------------
// One-time setup / teardown (all threads of both CTAs).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t g2_setup(const G2Smem& sm, int warp, int lane) {
    if (warp == G2_WARP_TMA && lane == 0) {
        for (int s = 0; s < G2_STAGES; ++s) { ptx::mbar_init(sm.full(s), 1); ptx::mbar_init(sm.empty(s), 1); }
        for (int a = 0; a < 2; ++a) { ptx::mbar_init(sm.tfull(a), 1); ptx::mbar_init(sm.tempty(a), 2 * G2_EPI_WARPS); }
        for (int q = 0; q < G2_NTI; ++q) { ptx::mbar_init(sm.ti_full(q), 1); ptx::mbar_init(sm.ti_empty(q), G2_TI_CONSUMERS); }
        ptx::st_shared_volatile_u32(sm.want(), 0u);
        for (int q = 0; q < G2_NTI; ++q) ptx::mbar_init(sm.cdone(q), 2 * G2_EPI_WARPS);
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
__device__ __forceinline__ void g2_teardown(uint32_t tmem_base, int warp) {
    ptx::tc_fence_before();
    ptx::cluster_sync();
    if (warp == G2_WARP_MMA) ptx::tmem_dealloc_pair(tmem_base, 512);
}

// Consumer side of the TileInfo ring: wait for record q, copy it to registers, release the ring entry.
// A stalled wait returns a record with valid == 0: the role leaves its loop. WARP = true: called by a whole warp
// (lane `release_lane` releases the entry); WARP = false: called by the single thread that runs a role.
template <bool WARP>
__device__ __forceinline__ TileInfo g2_take(const G2Smem& sm, int q, uint32_t ph, bool release_lane, volatile int* abort_flag) {
    TileInfo ti;
    if (!ptx::mbar_wait_patient(sm.ti_full(q), ph, abort_flag)) { ti.valid = 0; return ti; }      // record written with st.async: CTA-scope wait
    uint32_t* w = reinterpret_cast<uint32_t*>(&ti);
#pragma unroll
    for (int i = 0; i < 16; i += 4)
        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(w[i]), "=r"(w[i + 1]), "=r"(w[i + 2]), "=r"(w[i + 3]) : "r"(sm.tinfo(q) + 4u * i) : "memory");
    if (WARP) __syncwarp();
    if (release_lane) ptx::mbar_arrive_cluster_relaxed(ptx::mapa(sm.ti_empty(q), 0), w[0] ^ w[15]);
    return ti;
}

// ------------------------------------------------------------------------------------------------
// Finisher (one warp of the PEER CTA, which has no scheduler and no MMA issuer to run): per tile it waits until the
// epilogue warps of both CTAs have reported that their stores are in global memory, then `done(ti)` counts the tile
// and, for the last tile of a GEMM, runs the slot's transition. The epilogue warps never wait for the completion of
// their stores, for the counting atomic or for a transition: per tile that was a CTA-wide barrier, a bulk-store wait, a
// fence and an atomic round trip on the epilogue's path, more than the k-loop of a 560-wide tile.
// The ring entry is released only after the tile is complete, so the epilogue can never be a full ring ahead of it.
// ------------------------------------------------------------------------------------------------
template <typename Done>
__device__ __forceinline__ void g2_finisher(const G2Smem& sm, int lane, Done done, volatile int* abort_flag) {
    int q = 0; uint32_t tph = 0;
    for (;;) {
        const TileInfo ti = g2_take<true>(sm, q, tph, false, abort_flag);
        if (!ti.valid) {
            if (lane == 0) ptx::mbar_arrive_cluster(ptx::mapa(sm.ti_empty(q), 0));
            break;
        }
        if (!ptx::mbar_wait_cluster_patient(sm.cdone(q), tph, abort_flag)) break;
        if (lane == 0) {
            ptx::mbar_arrive_cluster(ptx::mapa(sm.ti_empty(q), 0));
            done(ti);
        }
        __syncwarp();
        if (++q == G2_NTI) { q = 0; tph ^= 1; }
    }
}

// ------------------------------------------------------------------------------------------------
// TMA producer (one warp per CTA). The whole warp runs the loop on warp-uniform values and ONE ELECTED lane issues: with
// `elect.sync` the compiler keeps the tensor-map addresses, coordinates and barrier addresses in uniform registers and the
// loads go out back to back. (With `if (lane == 0)` around the issue block every UTMALDG sat in a loop over the distinct
// values of its operands; the k-block then took ~650 cycles whatever the tile's width, the producer was busy 85 % of the
// time and the MMA warp waited for operands: profiles/r02_persist.md.)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void g2_producer(const G2Smem& sm, const CUtensorMap* maps, uint32_t rank, int lane, int want_lead, volatile int* abort_flag, int l2_load) {
    const uint64_t pol = ptx::l2_policy(l2_load);
    int stage = 0; uint32_t phase = 0;
    int q = 0; uint32_t tph = 0;
    uint32_t started = 0;                                                   // tiles that have reached their claim point
    const uint32_t full0 = ptx::mapa(sm.full(0), 0);                        // the leader's full barriers
    for (;;) {
        const TileInfo ti = g2_take<true>(sm, q, tph, lane == 0, abort_flag);
        if (++q == G2_NTI) { q = 0; tph ^= 1; }
        if (!ti.valid) break;
        ++started;
        ptx::fence_proxy_async();      // operands may have been written by generic stores of another CTA
        const CUtensorMap* map_a = maps + (size_t)ti.slot * NMAP + ti.a_buf;
        const CUtensorMap* map_b = maps + (size_t)ti.slot * NMAP + ti.b_buf;
        const int nkb = (ti.n16 + BK - 1) / BK;
        const int half = ti.bn >> 1;
        const int nbox = (half + 63) >> 6;
        const bool hh = (ti.valid & TI_HALF) != 0;                         // half-height tile: 64 rows of A per CTA
        const uint32_t bytes = 2u * ((hh ? G2_A_BYTES / 2 : G2_A_BYTES) + nbox * B_BOX_BYTES);     // both CTAs of the pair
        const int row0 = ti.m0 + (hh ? 64 : 128) * (int)rank;
        const int col0 = ti.n0 + half * (int)rank;
        const int kb_want = rank == 0 ? max(0, nkb - want_lead) : -1;
        // transposed tile: the A stage takes this CTA's 128 columns of B (two boxes), the B stage its bn / 2 rows of A
        const bool tr = (ti.valid & TI_TRANS) != 0;
        const int tcol0 = ti.n0 + 128 * (int)rank, trow0 = ti.m0 + half * (int)rank;
#pragma unroll 1
        for (int kb = 0; kb < nkb; ++kb) {
            if (!ptx::mbar_wait(sm.empty(stage), phase ^ 1, abort_flag)) return;
            if (tr) {
                if (ptx::elect_one()) {
                    if (kb == kb_want) ptx::st_shared_volatile_u32(sm.want(), started);
                    const uint32_t fb = full0 + 8u * stage;
                    if (rank == 0) ptx::mbar_expect_tx(sm.full(stage), bytes);
                    const uint32_t sa = sm.stage_a(stage), sb = sm.stage_b(stage);
                    const int k0 = kb * BK;
                    ptx::tma_load_2d_pair(sa, map_b, tcol0, k0, fb, pol);
                    ptx::tma_load_2d_pair(sa + 8192, map_b, tcol0 + 64, k0, fb, pol);
                    ptx::tma_load_2d_pair(sb, map_a, k0, trow0, fb, pol);
                    if (nbox > 1) ptx::tma_load_2d_pair(sb + B_BOX_BYTES, map_a, k0, trow0 + 64, fb, pol);
                }
            } else
            if (ptx::elect_one()) {
                if (kb == kb_want) ptx::st_shared_volatile_u32(sm.want(), started);   // the scheduler may claim the next tile now
                const uint32_t fb = full0 + 8u * stage;
                if (rank == 0) ptx::mbar_expect_tx(sm.full(stage), bytes);
                const uint32_t sa = sm.stage_a(stage), sb = sm.stage_b(stage);
                const int k0 = kb * BK;
                ptx::tma_load_2d_pair(sa, map_a, k0, row0, fb, pol);
                if (!hh) ptx::tma_load_2d_pair(sa + 8192, map_a, k0, row0 + 64, fb, pol);
                ptx::tma_load_2d_pair(sb, map_b, col0, k0, fb, pol);
                if (nbox > 1) ptx::tma_load_2d_pair(sb + B_BOX_BYTES, map_b, col0 + 64, k0, fb, pol);
            }
            __syncwarp();
            if (++stage == G2_STAGES) { stage = 0; phase ^= 1; }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// MMA issuer (one warp of the leader CTA; one elected lane issues, see g2_producer).
// The issue loop must stay well under the tensor-pipe time of a k-block (4 MMAs x ~120 cycles): the
// four MMAs of a full k-block go out as one asm block with the descriptors advanced by immediates
// (A: +32 B per 16 k inside the 128-byte swizzle row; B: +2048 B = 16 k-rows of 128 B).
// ------------------------------------------------------------------------------------------------
namespace ptx {
// 4 x (M = 256, N, K = 16) on one 64-k stage; acc0 = 0 overwrites the accumulator with the first MMA.
template <int SA = 2, int SB = 128>      // descriptor steps per 16 k (16-byte units): K-major operand 2, MN-major operand 128
__device__ __forceinline__ void umma_f16_pair_x4(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc0) {
    asm volatile(
        "{\n\t.reg .pred p, t;\n\t.reg .b64 a1, b1, a2, b2, a3, b3;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "setp.eq.b32 t, 0, 0;\n\t"
        "add.s64 a1, %1, %5;\n\tadd.s64 b1, %2, %6;\n\t"
        "add.s64 a2, %1, %7;\n\tadd.s64 b2, %2, %8;\n\t"
        "add.s64 a3, %1, %9;\n\tadd.s64 b3, %2, %10;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], a1, b1, %3, t;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], a2, b2, %3, t;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], a3, b3, %3, t;\n\t}\n"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc0),
          "n"(SA), "n"(SB), "n"(2 * SA), "n"(2 * SB), "n"(3 * SA), "n"(3 * SB) : "memory");
}
}  // namespace ptx

// mma_ns (nullable): [0] waiting for a tile record, [1] waiting for a free accumulator (the epilogue), [2] inside k-loops
// (operand waits + issue), summed over the leader CTAs, nanoseconds (three timer reads per tile).
__device__ __forceinline__ void g2_mma(const G2Smem& sm, uint32_t tmem_base, int lane, volatile int* abort_flag, unsigned long long* mma_ns) {
    unsigned long long t_take = 0, t_acc = 0, t_k = 0;
    int stage = 0; uint32_t phase = 0;
    int acc = 0; uint32_t acc_phase = 0;
    int q = 0; uint32_t tph = 0;
    // descriptors of stage 0; stage s adds s * G2_STAGE_BYTES / 16 to the address field
    const uint64_t da0 = make_smem_desc(sm.stage_a(0), 16, 1024);
    const uint64_t db0 = make_smem_desc(sm.stage_b(0), B_BOX_BYTES, 1024);
    // transposed tiles (TI_TRANS): the A stage holds columns of B (MN-major), the B stage rows of A (K-major)
    const uint64_t dat0 = make_smem_desc(sm.stage_a(0), B_BOX_BYTES, 1024);
    const uint64_t dbt0 = make_smem_desc(sm.stage_b(0), 16, 1024);
    for (;;) {
        const unsigned long long t0 = ptx::globaltimer_ns();
        const TileInfo ti = g2_take<true>(sm, q, tph, lane == 0, abort_flag);
        if (++q == G2_NTI) { q = 0; tph ^= 1; }
        if (!ti.valid) break;
        const unsigned long long t1 = ptx::globaltimer_ns();
        const int nkb = (ti.n16 + BK - 1) / BK;
        const int ktail = (ti.n16 - (nkb - 1) * BK) >> 4;          // 16-k slices of the last k-block (1..4)
        const bool tr = (ti.valid & TI_TRANS) != 0;
        const uint32_t idesc = make_idesc_f16((ti.valid & TI_HALF) ? 128 : 256, ti.bn) ^ (tr ? (3u << 15) : 0u);   // A MN-major, B K-major
        if (!ptx::mbar_wait_cluster(sm.tempty(acc), acc_phase ^ 1, abort_flag)) return;
        ptx::tc_fence_after();
        const unsigned long long t2 = ptx::globaltimer_ns();
        const uint32_t d_tmem = tmem_base + acc * 256;
#pragma unroll 1
        for (int kb = 0; kb < nkb; ++kb) {
            if (!ptx::mbar_wait(sm.full(stage), phase, abort_flag)) return;
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
                const uint64_t da = (tr ? dat0 : da0) + (uint64_t)(stage * (G2_STAGE_BYTES >> 4));
                const uint64_t db = (tr ? dbt0 : db0) + (uint64_t)(stage * (G2_STAGE_BYTES >> 4));
                if (kb < nkb - 1 || ktail == 4) {
                    if (!tr) ptx::umma_f16_pair_x4<2, 128>(d_tmem, da, db, idesc, kb != 0);
                    else ptx::umma_f16_pair_x4<128, 2>(d_tmem, da, db, idesc, kb != 0);
                } else {
                    const int sa = tr ? 128 : 2, sb = tr ? 2 : 128;
                    for (int k = 0; k < ktail; ++k)
                        ptx::umma_f16_pair(d_tmem, da + sa * k, db + sb * k, idesc, (kb | k) != 0);
                }
                ptx::umma_commit_pair(sm.empty(stage));
                if (kb == nkb - 1) ptx::umma_commit_pair(sm.tfull(acc));
            }
            __syncwarp();
            if (++stage == G2_STAGES) { stage = 0; phase ^= 1; }
        }
        if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        t_take += t1 - t0; t_acc += t2 - t1; t_k += ptx::globaltimer_ns() - t2;
    }
    if (mma_ns && lane == 0) { atomicAdd(&mma_ns[0], t_take); atomicAdd(&mma_ns[1], t_acc); atomicAdd(&mma_ns[2], t_k); }
}

// ------------------------------------------------------------------------------------------------
// Epilogue (warps 0..7 of each CTA): C = c_out * acc + beta * I, FP16 stores, fused squared
// residual || alpha_res A B - I ||_F^2 (the convergence test, C-7). Every warp reports to the finisher
// (g2_finisher) once its stores of the tile are in global memory.
//
// TI_MIRROR (symmetric products): only the tiles on and above the diagonal of the tile grid are
// multiplied; an off-diagonal tile also writes its transpose into the block below the diagonal (lanes of a warp are
// consecutive rows, so element j of every lane is a run of 32 consecutive FP16 of one row of C^T: one 64-byte store
// instruction per column) and its residual counts twice.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void st_mirror(__half* Ct /* &C[col_first][row] */, int ldc, const uint32_t* hp, int ncols) {
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        if (j < ncols) {
            const unsigned short v = (unsigned short)((j & 1) ? (hp[j >> 1] >> 16) : (hp[j >> 1] & 0xFFFFu));
            asm volatile("st.global.b16 [%0], %1;" ::"l"(Ct + (size_t)j * ldc), "h"(v) : "memory");
        }
    }
}

template <typename Eng>
__device__ __forceinline__ void g2_epilogue(const G2Smem& sm, uint32_t tmem_base, const Eng& e, __half* base,
                                            uint32_t rank, int warp, int lane, const CUtensorMap* maps, volatile int* abort_flag, int l2_store) {
    const uint64_t pol = ptx::l2_policy(l2_store);
    int acc = 0; uint32_t acc_phase = 0;
    int q = 0; uint32_t tph = 0;
    const uint32_t tempty0 = ptx::mapa(sm.tempty(0), 0);
    const int quarter = warp & 3, chalf = warp >> 2;
    const int g = quarter >> 1;                                    // row group (64 rows) of the TMA-store path
    bool stalled = false;
    for (;;) {
        const TileInfo ti = g2_take<true>(sm, q, tph, lane == 0, abort_flag);
        const uint32_t cdone_peer = ptx::mapa(sm.cdone(q), 1);
        if (++q == G2_NTI) { q = 0; tph ^= 1; }
        if (!ti.valid) break;
        const int n = ti.n, n16 = ti.n16;
        int ldc;
        __half* C = c_ptr(e, base, ti.slot, ti.c_buf, ldc);
        const bool ident = (ti.valid & TI_PLAIN) == 0;             // plain tiles: C = c_out acc, res = ||alpha_res acc||_F^2 (no identity)
        // full-height tile: the CTA's 128 TMEM lanes are 128 rows, every warp sees all bn columns; half-height tile
        // (M = 128 over the pair): lanes 0-63 and 64-127 are the same 64 rows with the left / right half of the columns
        const bool hh = (ti.valid & TI_HALF) != 0;
        // transposed tile: the lanes are COLUMNS of C (n0 + ...), the accumulator columns its rows m0 .. m0 + bn - 1; below,
        // "row" / "col" then name the lane / accumulator-column coordinate and only the stores swap them back
        const bool trans = (ti.valid & TI_TRANS) != 0;
        const int rbase = trans ? ti.n0 + 128 * (int)rank + quarter * 32
                        : hh ? ti.m0 + 64 * (int)rank + (quarter & 1) * 32 : ti.m0 + 128 * (int)rank + quarter * 32;   // first row of this warp
        const int row = rbase + lane;
        const int col0 = trans ? ti.m0 : hh ? ti.n0 + (quarter >> 1) * (ti.bn >> 1) : ti.n0;
        const int bn = hh ? ti.bn >> 1 : ti.bn;                        // columns this warp's lanes hold
        const float sa = ti.c_out;
        if (!ptx::mbar_wait_sleepy(sm.tfull(acc), acc_phase, abort_flag)) { stalled = true; break; }
        ptx::tc_fence_after();
        float rsum = 0.f, vsum = 0.f;
        uint32_t dep = 0;
        const bool symdiag = (ti.valid & TI_SYMDIAG) != 0;         // diagonal tile of a symmetric product
        const bool via_tma = ident && !hh;                         // full-height square GEMM tiles leave through shared memory and TMA stores
        float rsum2 = 0.f, vsum2 = 0.f;                            // residual terms of boxes that stand for their mirror image too
        if (via_tma) {
            // C leaves in 64 x 64 boxes: the four warps that hold rows [64 g, 64 g + 64) of the CTA's 128 rows and the two
            // 32-column halves of a box write it into a swizzled staging buffer; one thread hands it to the TMA unit, which
            // writes whole 128-byte lines (the row-per-thread register stores issue one request per 32 bytes and go
            // through the SM's load/store path, which the k-loop's ingest also needs). Two buffers per row group.
            // Symmetric products (TI_MIRROR / TI_SYMDIAG): a box above the diagonal is also written TRANSPOSED into the
            // second buffer and stored to the mirrored position (2-byte shared-memory stores, conflict-free under the
            // 128-byte swizzle; the transposed copy as 2-byte global stores cost 16 % of the Loewdin form's throughput);
            // a box on the diagonal is filled from its upper triangle, so the stored matrix is exactly symmetric; a box
            // below the diagonal is not stored at all.
            const int rbox = ((quarter & 1) << 5) + lane;
            const bool issuer = (quarter & 1) == 0 && chalf == 0 && lane == 0;
            const CUtensorMap* map_c = maps + (size_t)ti.slot * NMAP + ti.c_buf;
            const int nbx = (bn + 63) >> 6;
            const int brow = (trans ? ti.n0 : ti.m0) + 128 * (int)rank + 64 * g;     // first row of this group's boxes
            int bsel = 0;
            for (int kx = 0; kx < nbx; ++kx) {
                const int c = (kx << 6) + (chalf << 5);
                const int bcol = col0 + (kx << 6);                 // first column of the box
                // 0: plain box; 1: box above the diagonal of a symmetric product (stored and mirrored); 2: diagonal box;
                // 3: box below the diagonal (skipped). Uniform over the four warps of the group.
                // 4: box of a transposed tile (written transposed only).
                const int mode = trans ? 4 : (ti.valid & TI_MIRROR) ? 1 : !symdiag ? 0 : bcol > brow ? 1 : bcol == brow ? 2 : 3;
                if (mode == 3) continue;
                const uint32_t box = sm.stage_c(g, mode == 1 ? 0 : bsel), boxt = sm.stage_c(g, 1);
                if (issuer) { if (mode == 1) ptx::bulk_wait_read<0>(); else ptx::bulk_wait_read<1>(); }   // the stores that read these buffers are done with them
                asm volatile("bar.sync %0, 128;" ::"r"(3 + g) : "memory");
                float f[32];
                int ncols = 0;                                     // valid columns of this chunk (warp-uniform)
                if (c < bn && col0 + c < n16) {
                    uint32_t v[32];
                    ptx::tmem_ld_32x32(tmem_base + acc * 256 + ((uint32_t)(quarter * 32) << 16) + c, v);
                    ptx::tmem_ld_wait();
                    dep ^= v[0];
                    ncols = min(min(32, bn - c), n16 - (col0 + c));
                    const bool diag = (col0 + c < rbase + 32) && (col0 + c + 32 > rbase);
                    if (ncols == 32 && !diag) {
                        if (ti.want_res && row < n16) {
                            float vs = 0.f;
#pragma unroll
                            for (int j = 0; j < 32; ++j) { const float a = __uint_as_float(v[j]); vs = fmaf(a, a, vs); }
                            if (mode == 1) vsum2 += vs; else vsum += vs;
                        }
#pragma unroll
                        for (int j = 0; j < 32; ++j) f[j] = sa * __uint_as_float(v[j]);
                    } else {
                        float rs = 0.f;
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            const int col = col0 + c + j;
                            const float a = __uint_as_float(v[j]);
                            const float delta = (col == row && row < n) ? 1.f : 0.f;
                            const bool in = (j < ncols && row < n16);
                            const float d = in ? ti.alpha_res * a - delta : 0.f;      // pad rows / columns give exactly 0
                            rs = fmaf(d, d, rs);
                            f[j] = in ? ti.c_out * a + ti.beta * delta : 0.f;
                        }
                        if (mode == 1) rsum2 += rs; else rsum += rs;
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < 32; ++j) f[j] = 0.f;
                }
                uint32_t hp[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) { __half2 h = __floats2half2_rn(f[2 * j], f[2 * j + 1]); hp[j] = *reinterpret_cast<uint32_t*>(&h); }
                if (mode == 4) {
                    ptx::st_box_col(box, rbox, chalf << 5, hp);
                } else if (mode != 2) {
                    ptx::st_box_row(box, rbox, chalf << 2, hp);
                    if (mode == 1) ptx::st_box_col(boxt, rbox, chalf << 5, hp);
                } else {
                    ptx::st_box_sym(box, rbox, chalf << 5, hp);
                }
                ptx::fence_proxy_async_smem();
                asm volatile("bar.sync %0, 128;" ::"r"(3 + g) : "memory");
                if (issuer) {
                    if (mode == 4) {
                        ptx::tma_store_2d(map_c, brow, bcol, box, pol);
                    } else if (brow < n16) {                       // boxes below the matrix are padding
                        ptx::tma_store_2d(map_c, bcol, brow, box, pol);
                        if (mode == 1) ptx::tma_store_2d(map_c, brow, bcol, boxt, pol);
                    }
                    ptx::bulk_commit();
                }
                if (mode != 1) bsel ^= 1;
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_cluster_relaxed(tempty0 + 8u * acc, dep);     // the accumulator is free
            if (issuer) ptx::bulk_wait<0>();                       // the boxes of this tile are in global memory
        } else
        for (int c = chalf * 32; c < bn; c += 64) {
            if (col0 + c >= n16) break;                            // warp-uniform
            uint32_t v[32];
            ptx::tmem_ld_32x32(tmem_base + acc * 256 + ((uint32_t)(quarter * 32) << 16) + c, v);
            ptx::tmem_ld_wait();
            dep ^= v[0];
            if (ti.valid & TI_F32OUT) {                            // P[row, 0..31] = acc, FP32 (a6: D columns are formed from FP32)
                if (c == 0 && row < n16) {
                    float4* prow = reinterpret_cast<float4*>(pcols_ptr(e, ti.slot) + (size_t)row * PCW);
#pragma unroll
                    for (int j = 0; j < PCW; j += 4)
                        prow[j >> 2] = make_float4(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]), __uint_as_float(v[j + 3]));
                }
                continue;
            }
            const int gc0 = col0 + c;                              // first column of this chunk
            __half* crow = C + (size_t)row * ldc + gc0;
            const int cw = min(min(32, bn - c), n16 - gc0);        // 16 or 32 valid columns (warp-uniform)
            const bool diag = (gc0 < rbase + 32) && (gc0 + 32 > rbase);
            float f[32];
            if (cw == 32 && !diag) {
                // interior chunk: C = (sgn alpha) acc, residual term alpha^2 acc^2 (no identity entries here)
                if (row < n16) {
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const float a = __uint_as_float(v[j]);
                        vsum = fmaf(a, a, vsum);
                        f[j] = sa * a;
                    }
                }
            } else if (row < n16) {
#pragma unroll
                for (int j = 0; j < 32; ++j) {
                    const int col = gc0 + j;
                    const float a = __uint_as_float(v[j]);
                    const float delta = (col == row && row < n && ident) ? 1.f : 0.f;
                    const float d = j < cw ? ti.alpha_res * a - delta : 0.f;   // pad rows / columns give exactly 0
                    rsum = fmaf(d, d, rsum);
                    f[j] = ti.c_out * a + ti.beta * delta;
                }
            }
            if (row < n16) {
                if (!symdiag) {
#pragma unroll
                    for (int j = 0; j < 32; j += 16)
                        if (j < cw) st_half16(crow + j, f + j);
                } else if (gc0 >= rbase + 32) {
                    // diagonal tile of a symmetric product, chunk above the diagonal: stored and mirrored; the chunks below
                    // the diagonal are not stored (their mirror images are), so the stored matrix is exactly symmetric
                    uint32_t hp[16];
#pragma unroll
                    for (int j = 0; j < 16; ++j) { __half2 h = __floats2half2_rn(f[2 * j], f[2 * j + 1]); hp[j] = *reinterpret_cast<uint32_t*>(&h); }
#pragma unroll
                    for (int j = 0; j < 32; j += 16)
                        if (j < cw) st_half16(crow + j, f + j);
                    st_mirror(C + (size_t)gc0 * ldc + row, ldc, hp, cw);
                } else if (gc0 + 32 > rbase) {
                    // chunk that holds diagonal elements: element by element, upper triangle stored and mirrored
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const int col = gc0 + j;
                        if (j < cw && col >= row) {
                            const __half h = __float2half_rn(f[j]);
                            crow[j] = h;
                            if (col > row) C[(size_t)col * ldc + row] = h;
                        }
                    }
                }
            }
        }
        if (!via_tma) {
            ptx::tc_fence_before();
            ptx::fence_proxy_async();      // C is read next through the async proxy (TMA), possibly by another CTA
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_cluster_relaxed(tempty0 + 8u * acc, dep);
        }
        if (ti.want_res) {
            rsum = fmaf(ti.alpha_res * ti.alpha_res, vsum, rsum) + 2.f * fmaf(ti.alpha_res * ti.alpha_res, vsum2, rsum2);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) rsum += __shfl_xor_sync(0xffffffffu, rsum, o);
            if (lane == 0 && rsum != 0.f) atomicAdd(&e.slots[ti.slot].res_acc, rsum);
        }
        // this warp's stores of the tile are in global memory (the TMA stores of its row group: the issuer waited for them)
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_cluster(cdone_peer);
        if (++acc == 2) { acc = 0; acc_phase ^= 1; }
    }
    if (stalled) {
        // a warp that gives up on a stalled wait releases the named barriers its peers may be waiting at (they stall and
        // leave at their next wait)
        asm volatile("bar.arrive %0, 128;" ::"r"(3 + g) : "memory");
    }
}

}  // namespace nolsm
