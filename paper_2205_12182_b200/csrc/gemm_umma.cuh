// Grouped, variable-size FP16 x FP16 -> FP32 GEMM for sm_100a: TMA loads into 128B-swizzled shared
// memory, tcgen05.mma (kind::f16, cta_group::1, M=128, N<=256) accumulating in TMEM, double-buffered
// TMEM accumulators drained by four epilogue warps with tcgen05.ld.
//
// This is the GEMM "C = alpha A B + beta C" the paper counts as 2n^3 FLOP inside
// the matrix iterations (Eq. 6; Schulz inverse, ref [14] PAPER.md:L217). All three
// matrices are row-major, so A is a K-major operand and B an MN-major operand of the UMMA; X*X
// therefore needs no transposed copy of X.
//
// Persistent kernel: grid = #SMs, each CTA walks the round's tile list (all slots that take part in
// this launch, nolsm_device.cuh) with stride gridDim.x; the tile count is read from device memory.
// Warp roles: warp 0 = TMA producer, warp 1 = TMEM allocator + MMA issuer, warps 2..5 = epilogue.
#pragma once
#include "nolsm_device.cuh"

namespace nolsm {

constexpr int UMMA_STAGES = 4;
constexpr int UMMA_THREADS = 192;
constexpr int A_STAGE_BYTES = BM * BK * 2;          // 16 KB
constexpr int B_BOX_BYTES = BK * 64 * 2;            // one 64(n) x 64(k) box = 8 KB
constexpr int B_STAGE_BYTES = 4 * B_BOX_BYTES;      // up to N = 256
constexpr int STAGE_BYTES = A_STAGE_BYTES + B_STAGE_BYTES;
constexpr int UMMA_SMEM_BYTES = UMMA_STAGES * STAGE_BYTES + 1024 /*align*/ + 256 /*barriers*/;
constexpr uint32_t SPIN_LIMIT = 1u << 28;

namespace ptx {

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ bool elect_one() {
    uint32_t pred = 0;
    asm volatile(
        "{\n\t.reg .b32 rx;\n\t.reg .pred px;\n\t"
        "elect.sync rx|px, 0xffffffff;\n\t"
        "selp.b32 %0, 1, 0, px;\n\t}\n"
        : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}\n"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// Bounded wait: a protocol bug traps (the launch fails with an error) instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > SPIN_LIMIT) __trap();
    }
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void umma_f16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}\n"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// 32 lanes x 32 columns of fp32: thread l of the warp receives columns [c, c+32) of TMEM lane (base + l).
__device__ __forceinline__ void tmem_ld_32x32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

}  // namespace ptx

// Shared-memory matrix descriptor (tcgen05 "smem descriptor"): start address, leading / stride byte
// offsets (all >> 4), version 1 (Blackwell), layout type 2 = SWIZZLE_128B.
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
// Instruction descriptor for kind::f16: FP32 accumulate, FP16 A and B, A K-major, B MN-major.
__device__ __forceinline__ uint32_t make_idesc_f16(int m, int n) {
    uint32_t d = 0;
    d |= 1u << 4;                    // D format: F32
    d |= 0u << 7;                    // A format: F16
    d |= 0u << 10;                   // B format: F16
    d |= 0u << 15;                   // A major: K
    d |= 1u << 16;                   // B major: MN
    d |= (uint32_t)(n >> 3) << 17;
    d |= (uint32_t)(m >> 4) << 24;
    return d;
}

struct UmmaArgs {
    Engine e;
    const CUtensorMap* maps;    // [S][NBUF]: cap x cap, row pitch ld, box 64 x 64, SWIZZLE_128B
    __half* base;               // workspace base
    int launch;                 // 0 or 1: which op table of the round
};

__device__ __forceinline__ void st_half8(__half* p, const float* v) {
    __half2 h0 = __floats2half2_rn(v[0], v[1]);
    __half2 h1 = __floats2half2_rn(v[2], v[3]);
    __half2 h2 = __floats2half2_rn(v[4], v[5]);
    __half2 h3 = __floats2half2_rn(v[6], v[7]);
    uint4 u;
    u.x = *reinterpret_cast<uint32_t*>(&h0);
    u.y = *reinterpret_cast<uint32_t*>(&h1);
    u.z = *reinterpret_cast<uint32_t*>(&h2);
    u.w = *reinterpret_cast<uint32_t*>(&h3);
    *reinterpret_cast<uint4*>(p) = u;
}

__global__ void __launch_bounds__(UMMA_THREADS, 1) gemm_umma_kernel(const __grid_constant__ UmmaArgs args) {
    extern __shared__ uint8_t smem_raw[];
    const Engine& e = args.e;
    const SlotOp* ops = e.ops + args.launch * e.S;
    const int ntiles = e.ntiles[args.launch];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + UMMA_STAGES * STAGE_BYTES;
    // barrier layout (8 B each): full[S], empty[S], tmem_full[2], tmem_empty[2], then tmem ptr
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (UMMA_STAGES + s); };
    auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * UMMA_STAGES + s); };
    auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * UMMA_STAGES + 2 + s); };
    const uint32_t tmem_ptr_addr = bar_base + 8u * (2 * UMMA_STAGES + 4);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    if ((int)blockIdx.x >= ntiles) return;           // whole CTA idle this launch (uniform)

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < UMMA_STAGES; ++s) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
        for (int s = 0; s < 2; ++s) { ptx::mbar_init(tfull_bar(s), 1); ptx::mbar_init(tempty_bar(s), 4); }
        ptx::fence_mbar_init();
    }
    if (warp == 1) ptx::tmem_alloc(tmem_ptr_addr, 512);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_addr));

    if (warp == 0) {
        // ================= TMA producer =================
        if (lane == 0) {
            int stage = 0; uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                const int slot = find_slot(ops, e.S, tile);
                const SlotOp op = ops[slot];
                const Slot& sl = e.slots[slot];
                const int n16 = sl.n16, bn = sl.bn, ntn = sl.ntn;
                const int t = tile - op.tile_start;
                const int tm = t / ntn, tn = t - tm * ntn;
                const CUtensorMap* map_a = args.maps + (size_t)slot * NBUF + op.a_buf;
                const CUtensorMap* map_b = args.maps + (size_t)slot * NBUF + op.b_buf;
                const int nkb = (n16 + BK - 1) / BK;
                const int nbox = (bn + 63) >> 6;
                const uint32_t bytes = A_STAGE_BYTES + nbox * B_BOX_BYTES;
                for (int kb = 0; kb < nkb; ++kb) {
                    ptx::mbar_wait(empty_bar(stage), phase ^ 1);
                    const uint32_t sa = smem_base + stage * STAGE_BYTES;
                    const uint32_t sb = sa + A_STAGE_BYTES;
                    ptx::mbar_expect_tx(full_bar(stage), bytes);
                    ptx::tma_load_2d(sa, map_a, kb * BK, tm * BM, full_bar(stage));
                    ptx::tma_load_2d(sa + 8192, map_a, kb * BK, tm * BM + 64, full_bar(stage));
                    for (int q = 0; q < nbox; ++q)
                        ptx::tma_load_2d(sb + q * B_BOX_BYTES, map_b, tn * bn + q * 64, kb * BK, full_bar(stage));
                    if (++stage == UMMA_STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ================= MMA issuer =================
        int stage = 0; uint32_t phase = 0;
        int acc = 0; uint32_t acc_phase = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const int slot = find_slot(ops, e.S, tile);
            const Slot& sl = e.slots[slot];
            const int n16 = sl.n16;
            const int nkb = (n16 + BK - 1) / BK;
            const uint32_t idesc = make_idesc_f16(BM, sl.bn);
            ptx::mbar_wait(tempty_bar(acc), acc_phase ^ 1);
            ptx::tc_fence_after();
            const uint32_t d_tmem = tmem_base + acc * 256;
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(full_bar(stage), phase);
                ptx::tc_fence_after();
                if (lane == 0) {
                    const uint32_t sa = smem_base + stage * STAGE_BYTES;
                    const uint32_t sb = sa + A_STAGE_BYTES;
                    int k16 = (n16 - kb * BK) >> 4;
                    k16 = k16 > 4 ? 4 : k16;
                    for (int k = 0; k < k16; ++k) {
                        const uint64_t da = make_smem_desc(sa + k * 32, 16, 1024);
                        const uint64_t db = make_smem_desc(sb + k * 2048, B_BOX_BYTES, 1024);
                        ptx::umma_f16(d_tmem, da, db, idesc, (kb | k) != 0);
                    }
                    ptx::umma_commit(empty_bar(stage));
                    if (kb == nkb - 1) ptx::umma_commit(tfull_bar(acc));
                }
                __syncwarp();
                if (++stage == UMMA_STAGES) { stage = 0; phase ^= 1; }
            }
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
    } else {
        // ================= epilogue (warps 2..5) =================
        const int q = warp & 3;                       // TMEM lane group this warp may access
        int acc = 0; uint32_t acc_phase = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const int slot = find_slot(ops, e.S, tile);
            const SlotOp op = ops[slot];
            const Slot& sl = e.slots[slot];
            const int n = sl.n, n16 = sl.n16, bn = sl.bn, ntn = sl.ntn;
            const int t = tile - op.tile_start;
            const int tm = t / ntn, tn = t - tm * ntn;
            __half* C = args.base + buf_off(e, slot, op.c_buf);
            const int row = tm * BM + q * 32 + lane;
            const int col0 = tn * bn;
            ptx::mbar_wait(tfull_bar(acc), acc_phase);
            ptx::tc_fence_after();
            float rsum = 0.f;
            for (int c = 0; c < bn; c += 32) {
                if (col0 + c >= n16) break;                        // warp-uniform
                uint32_t v[32];
                ptx::tmem_ld_32x32(tmem_base + acc * 256 + ((uint32_t)(q * 32) << 16) + c, v);
                ptx::tmem_ld_wait();
                if (row < n16) {
                    float f[32];
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const int col = col0 + c + j;
                        const float x = op.alpha * __uint_as_float(v[j]);
                        const float delta = (col == row && row < n) ? 1.f : 0.f;
                        if (op.want_res) {                             // pad rows / columns contribute exactly 0
                            const float d = (c + j < bn && col < n16) ? x - delta : 0.f;
                            rsum += d * d;
                        }
                        f[j] = op.sgn * x + op.beta * delta;
                    }
                    __half* crow = C + (size_t)row * e.ld + col0 + c;
                    // bn and n16 are multiples of 16: the valid part of this chunk is 16 or 32 columns
                    const int cw = min(min(32, bn - c), n16 - (col0 + c));
#pragma unroll
                    for (int j = 0; j < 32; j += 8)
                        if (j < cw) st_half8(crow + j, f + j);
                }
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(tempty_bar(acc));
            if (op.want_res) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) rsum += __shfl_xor_sync(0xffffffffu, rsum, o);
                if (lane == 0 && rsum != 0.f) atomicAdd(&e.slots[slot].res_acc, rsum);
            }
            // all four epilogue warps done with this tile -> one thread reports it
            asm volatile("bar.sync 1, 128;" ::: "memory");
            if (warp == 2 && lane == 0) tile_finished(e, slot, op);
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem_base, 512);
}

}  // namespace nolsm
