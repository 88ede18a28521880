// Persistent engine: the whole hot path a1-a7 of one nolsm_density_matrix call in ONE kernel launch.
//
// grid = one CTA per SM in clusters of four (two CTA pairs that share the A operand, gemm4sm.cuh); every CTA runs
//   warps 0-10   the grouped tcgen05 GEMM pipeline of gemm2sm.cuh (epilogue x 8, tile scheduler, TMA
//                producer, MMA issuer), fed from a device-side claim table instead of a static tile list;
//   warps 11-14  a SIDE GROUP that executes the O(n^2) steps of the path as small tasks: gather
//                (PAPER.md:L56, L60), the closed-form first Schulz step, and D columns + scatter +
//                energy (Eq. 4).
// The spectral scalings (rho(S_sub) for the Schulz start, rho(A_sub) for X0 = A / rho, C-6)
// come from a BLOCK power iteration with 16 vectors that runs as 256 x 16 GEMM tiles in the same
// pipeline (V <- alpha M V, Frobenius norm of the product from the fused residual reduction).
//
// A slot (nolsm_device.cuh) holds one atom submatrix. At any time a slot has at most ONE live piece of
// work: a GEMM op (claim word gclaim[slot] = tiles << 20 | next tile) or a side task (sclaim[slot] =
// kind << 28 | chunks << 14 | next chunk). Tiles / chunks are claimed with one atomicAdd; the thread
// that completes the last tile / chunk runs the slot's transition (convergence test, C-7) and
// installs the next piece of work, or refills the slot with the next atom. Schedulers scan the claim
// tables in slot order, so only as many slots as the GPU can keep busy are active at once and the
// iterates of the active slots stay resident in L2 from one GEMM to the next. The host launches the
// kernel once and waits.
//
// Cross-CTA data flow: GEMM outputs are written with generic stores and read back by TMA (async proxy)
// of other CTAs: writers fence (fence.proxy.async, __threadfence) before the completing atomic; readers
// fence.proxy.async after the claim. Slot state is read and written with .cg accesses (L1 is not
// coherent across SMs).
#pragma once
#include "gemm4sm.cuh"
#include "kernels.cuh"

namespace nolsm {

constexpr int P_SIDE_WARPS = 4;
constexpr int P_SIDE_THREADS = P_SIDE_WARPS * 32;
constexpr int P_THREADS = G2_CTRL_THREADS + P_SIDE_THREADS;
constexpr int P_SIDE_SMEM = 60 * 1024;
constexpr int P_SMEM_BYTES = G2_SMEM_BYTES + P_SIDE_SMEM;
constexpr int P_MAX_CAP = 4096;
constexpr int P_GATHER_ROWATOMS = 4;            // row-atoms of N(i) per gather chunk (at most)

enum SideKind { SK_NONE = 0, SK_REFILL, SK_GATHER, SK_SCHULZ1, SK_DCOLS };

// counters written by the kernel (unsigned long long each)
enum { PC_TILES = 0, PC_SCHED_IDLE_NS, PC_SCHED_BUSY_NS, PC_OVERSHOOT, PC_T_START, PC_T_END,
       PC_SIDE_NS,            // + kind
       PC_SIDE_BYTES = PC_SIDE_NS + 8,   // + kind (algorithmic bytes)
       PC_SIDE_TASKS = PC_SIDE_BYTES + 8,
       PC_LEN = PC_SIDE_TASKS + 8 };

struct __align__(16) PSlot {      // 160 bytes
    int atom, n, n16, pos, nbi, ntm, ntn, nset;                     // geometry (written at refill)
    int op_kind, a_buf, b_buf, c_buf;                               // live GEMM op: C = c_out A B + beta I, residual of alpha_res A B
    float c_out, alpha_res, beta; int want_res;
    int inv_iters, sign_iters, conv, xcur, ycur, status, gemm_count, tiles_done;
    float res_acc, res_prev, res_last, rho_s, rho_a, alpha1, alpha2; int side_done;
    int pow_step; float pow_norm2, pow_alpha; int resume;           // block power iteration state; resume: which token phase comes next
    int noboost, unit, mptr, mend;                                  // noboost: the scaled steps are over for this matrix; unit and its members
                                                                    // [mptr, mend) still to be served (atom / pos / nbi describe member mptr)
};

struct PEngine {
    PSlot* slots;
    unsigned long long* gclaim;   // [S] GEMM claim words
    unsigned int* sclaim;         // [S] side-task claim words
    int S, cap, ld;
    long long bufsz, slotsz;
    float tol_inv, tol_sign, mu, safety_s, safety_a;
    int max_inv, max_sign, p_s, p_a;
    int gather_rowatoms, schulz_chunks, dcols_chunks;   // row-atoms of N(i) per gather chunk; chunks of the other tasks
    int* next_atom; int a_end, total;                 // feed position, its end, units of this call
    const int* feed;              // feed position -> unit id (nullptr: the position is the unit id)
    int atom_lo, atom_hi;         // only members inside [atom_lo, atom_hi) get their columns of D (nolsm_density_matrix_range)
    int* finished;
    int* heavy;                   // [1] slots inside the GEMM-heavy phases INV .. SIGN right now (at most g_max)
    int* parked;                  // [S] 1 = the slot finished its first Schulz step and waits for a heavy token
    int g_max, want_lead, dbg;
    int tma_store;                // 1: square GEMM tiles leave through shared-memory boxes and TMA stores
    int split_tokens;             // 1: the heavy token is returned for the rho(A) power iteration and taken again for the sign phase
    int gather_prefetch;          // 1: the gather task prefetches a row-atom's source blocks into L2 before staging them
    int half_tiles;               // 1: half-height (M = 128) tiles for a last row block of at most 128 rows
    int tile_n;                   // columns of a pair tile (256; 128 halves a GEMM's latency at more L2 traffic per FLOP)
    const signed char* die_of_sm; // [256] L2 die of every SM (0 / 1), or all -1: no die affinity (see k_die_probe)
    int ndie;                     // 2: slot s is served only by SMs of die s & 1 and heavy tokens are per die; 1: no affinity
    int ctas;                     // CTAs per cluster of the running kernel: 2 (pair tiles, gemm2sm.cuh) or 4 (A shared by two pairs, gemm4sm.cuh)
    int n_sched; float alpha_sched[16];   // scaled Newton-Schulz: alpha_k of sign iteration k < n_sched (1 afterwards)
    volatile int* abort_flag;     // device word; the host sets it (copy on another stream) to stop a kernel that overran its time limit
    unsigned long long* ctr;      // [PC_LEN]
    AtomArrays at;                // results are indexed by unit
    const int* udim;              // [n_units] dimension of the unit's matrix
    const int* upos;              // [n_atoms] first column of atom i inside its unit's matrix
    const int* adim;              // [n_atoms] dim N(i): rows of D written for atom i
    SysView sv;
    const void *S_vals, *H_vals; int val_f64;
    void* D_vals; int d_f64;
    double* e_atom;
    double* q_atom;               // [n_atoms] electron-count partials sum_j <D_ji, S_ji> (Tr(D S))
    const CUtensorMap* maps;
    __half* base;
    float* pcols;                 // [S][cap][PCW] FP32: X Y[:, cols(i)] of the slot's atom (OP_DCOLS)
};

__device__ __forceinline__ long long buf_off(const PEngine& e, int slot, int buf) {
    return (long long)slot * e.slotsz + (long long)buf * e.bufsz;
}
// Buffers 0..NBUF-1: the slot's square buffers (leading dimension ld). Buffers NBUF, NBUF+1: the slot's
// two vector blocks (cap x VLD, the first NVC columns are used); they follow the S slots in the workspace.
__device__ __forceinline__ __half* c_ptr(const PEngine& e, __half* base, int slot, int buf, int& ldc) {
    if (buf < NBUF) { ldc = e.ld; return base + buf_off(e, slot, buf); }
    ldc = VLD;
    return base + (long long)e.S * e.slotsz + ((long long)slot * 2 + (buf - NBUF)) * ((long long)e.cap * VLD);
}

__device__ __forceinline__ float* pcols_ptr(const PEngine& e, int slot) { return e.pcols + (size_t)slot * e.cap * PCW; }

// L2 die of the SM this CTA runs on (-1: no affinity). B200 is two dies, each with half of the SMs and half of
// L2; a line that SMs of both dies read is kept in both halves, so iterates shared across dies see only half of
// the 126 MB. With affinity a slot's buffers are touched by the SMs of one die only.
__device__ __forceinline__ int p_my_die(const PEngine& e) {
    if (e.ndie != 2) return -1;
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    return (int)e.die_of_sm[smid & 255u];
}

// Die probe: every CTA times dependent L2-hit loads (ld.global.cg chain) of NPROBE lines that lie 2 KB apart and
// records the best time per (SM, line). A line is homed in one die; the SMs of that die see it ~25 cycles sooner.
// The host turns the per-line near / far pattern into the SM -> die table.
constexpr int NPROBE = 16;
__global__ void __launch_bounds__(32) k_die_probe(const unsigned long long* lines, unsigned int* best /*[256][NPROBE]*/) {
    if (threadIdx.x != 0) return;
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    for (int l = 0; l < NPROBE; ++l) {
        const unsigned long long* p = lines + (size_t)l * 256;       // 2 KB apart
        unsigned long long v = 0;
        for (int i = 0; i < 8; ++i) asm volatile("ld.global.cg.u64 %0, [%1];" : "=l"(v) : "l"(p + v) : "memory");   // warm (lines hold 0)
        const long long t0 = clock64();
        for (int i = 0; i < 64; ++i) asm volatile("ld.global.cg.u64 %0, [%1];" : "=l"(v) : "l"(p + v) : "memory");
        const long long t1 = clock64();
        atomicMin(&best[(smid & 255u) * NPROBE + l], (unsigned)((t1 - t0) + (long long)v));
    }
}

namespace pl {
__device__ __forceinline__ unsigned long long gtime() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void side_sync() { asm volatile("bar.sync 2, %0;" ::"n"(P_SIDE_THREADS) : "memory"); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ float dot8(const uint4& m, const float4& x0, const float4& x1) {
    const __half2* h = reinterpret_cast<const __half2*>(&m);
    const float2 a = __half22float2(h[0]), b = __half22float2(h[1]), c = __half22float2(h[2]), d = __half22float2(h[3]);
    float s = a.x * x0.x;
    s = fmaf(a.y, x0.y, s); s = fmaf(b.x, x0.z, s); s = fmaf(b.y, x0.w, s);
    s = fmaf(c.x, x1.x, s); s = fmaf(c.y, x1.y, s); s = fmaf(d.x, x1.z, s); s = fmaf(d.y, x1.w, s);
    return s;
}
}  // namespace pl

// ------------------------------------------------------------------------------------------------
// Installing work on a slot (one thread; the slot has no other live work at that moment).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void p_install_side(const PEngine& e, int slot, int kind, int chunks) {
    __threadfence();
    *(volatile unsigned int*)&e.sclaim[slot] = ((unsigned)kind << 28) | ((unsigned)chunks << 14);
}

// Scaling alpha_k of sign iteration k (C-6b): X_{k+1} = 1/2 (alpha X_k)(3I - (alpha X_k)^2).
__device__ __forceinline__ float p_sign_alpha(const PEngine& e, const PSlot* s, int k) {
    return (k < e.n_sched && !__ldcg(&s->noboost)) ? e.alpha_sched[k] : 1.f;
}

__device__ __forceinline__ void p_install_gemm(const PEngine& e, int slot, int kind) {
    PSlot* s = &e.slots[slot];
    const int xcur = __ldcg(&s->xcur), ycur = __ldcg(&s->ycur);
    const int k = __ldcg(&s->sign_iters);
    const bool first = k == 0;
    int a = 0, b = 0, c = 0, want = 0;
    float c_out = 1.f, alpha_res = 1.f, beta = 0.f;
    switch (kind) {
        case OP_INV_G1: a = 0; b = ycur; c = 4; c_out = -1.f; beta = 2.f; want = 1; break;       // R = 2I - S Y
        case OP_INV_G2: a = ycur; b = 4; c = 5 - ycur; break;                                       // Y <- Y R
        case OP_AMAT: a = ycur; b = 1; c = 0; beta = -e.mu; break;                                  // A = Y H0 - mu I
        case OP_SIGN_G1: {                                                                          // T = 3I - alpha^2 X^2
            const float al = p_sign_alpha(e, s, k);
            alpha_res = first ? __ldcg(&s->alpha1) : 1.f;                                           // X0 = A / rho is never stored
            a = xcur; b = xcur; c = 4; c_out = -al * al * alpha_res; beta = 3.f; want = 1;
        } break;
        case OP_SIGN_G2: {                                                                          // X <- alpha/2 X T
            const float al = p_sign_alpha(e, s, k);
            a = xcur; b = 4; c = 1 - xcur; c_out = al * (first ? __ldcg(&s->alpha2) : 0.5f);
        } break;
        case OP_POW_S:
        case OP_POW_A: {                                                                            // V <- alpha M V
            const int st = __ldcg(&s->pow_step);
            a = 0; b = st == 0 ? NMAP - 1 : NBUF + ((st - 1) & 1); c = NBUF + (st & 1);
            c_out = alpha_res = __ldcg(&s->pow_alpha); want = 1;
        } break;
        case OP_DCOLS: a = xcur; b = ycur; c = 0; break;                                           // P = X Y[:, cols(i)]
        default: break;
    }
    __stcg(reinterpret_cast<int4*>(&s->op_kind), make_int4(kind, a, b, c));
    __stcg(reinterpret_cast<float4*>(&s->c_out), make_float4(c_out, alpha_res, beta, __int_as_float(want)));
    const bool pow = kind == OP_POW_S || kind == OP_POW_A || kind == OP_DCOLS;       // one 16-column tile per 256 rows
    const unsigned long long tiles = (unsigned long long)(__ldcg(&s->ntm) * (pow ? 1 : __ldcg(&s->ntn)));
    __threadfence();
    *(volatile unsigned long long*)&e.gclaim[slot] = tiles << 20;
}

// Starts the block power iteration on buffer 0 (S_sub or A_sub): V0 = the shared +-1 start block.
__device__ __forceinline__ void p_start_power(const PEngine& e, int slot, int kind) {
    PSlot* s = &e.slots[slot];
    __stcg(&s->pow_step, 0);
    __stcg(&s->pow_norm2, (float)NVC * (float)__ldcg(&s->n));
    __stcg(&s->pow_alpha, 1.f);
    p_install_gemm(e, slot, kind);
}

// L2 residency: a slot's iterates (X, T, Y: ~3-4 n^2 FP16) are re-read by every GEMM of its chain, so only
// as many slots as fit in L2 together may be inside the heavy phases (Schulz iterations .. sign iterations)
// at once. A slot that is ready to enter takes a token or parks; a slot that leaves hands its token to a
// parked slot (and installs that slot's first GEMM) or returns it.
// A slot takes a token twice: for the Schulz iterations .. A = S^-1 H0 (resume == 0) and, after the power iteration for
// rho(A) - nine dependent 16-column tile passes that would hold the token idle - for the sign iterations (resume == 1).
__device__ __forceinline__ void p_enter_heavy_now(const PEngine& e, int slot) {
    PSlot* s = &e.slots[slot];
    if (__ldcg(&s->resume) == 0) {
        __stcg(&s->inv_iters, 1);
        __stcg(&s->ycur, 2);
        p_install_gemm(e, slot, OP_INV_G1);
    } else {
        p_install_gemm(e, slot, OP_SIGN_G1);
    }
}
// With die affinity (ndie == 2) slot s belongs to die s & 1: tokens are counted per die (g_max each).
__device__ __forceinline__ void p_enter_heavy(const PEngine& e, int slot) {
    int* heavy = e.heavy + (e.ndie == 2 ? (slot & 1) : 0);
    if (atomicAdd(heavy, 1) < e.g_max) { p_enter_heavy_now(e, slot); return; }
    atomicSub(heavy, 1);
    __threadfence();
    atomicExch(&e.parked[slot], 1);
    __threadfence();
    // a token may have been returned between the failed attempt and the parking: try once more
    if (atomicAdd(heavy, 1) < e.g_max) {
        if (atomicCAS(&e.parked[slot], 1, 0) == 1) { p_enter_heavy_now(e, slot); return; }
        // a leaving slot admitted this one meanwhile (with its own token)
    }
    atomicSub(heavy, 1);
}
__device__ __forceinline__ void p_leave_heavy(const PEngine& e, int slot) {
    const int step = e.ndie == 2 ? 2 : 1;
    for (int s = e.ndie == 2 ? (slot & 1) : 0; s < e.S; s += step) {
        if (*(volatile int*)&e.parked[s] == 1 && atomicCAS(&e.parked[s], 1, 0) == 1) {
            __threadfence();
            p_enter_heavy_now(e, s);          // the token changes hands
            return;
        }
    }
    atomicSub(e.heavy + (e.ndie == 2 ? (slot & 1) : 0), 1);
}

// Takes the next atom of the feed into the slot and installs its gather (phase NEW). Returns false when
// the feed is exhausted (the slot stays free).
__device__ __forceinline__ bool p_refill(const PEngine& e, int slot) {
    if (*(volatile int*)e.next_atom >= e.a_end) return false;
    const int fpos = atomicAdd(e.next_atom, 1);                         // a unit of the feed
    if (fpos >= e.a_end) return false;
    const int a = e.feed ? e.feed[fpos] : fpos;
    PSlot* s = &e.slots[slot];
    const int n = e.udim[a], n16 = (n + 15) & ~15;
    int ntm, ntn;
    choose_tiling(n16, ntm, ntn);
    if (e.ctas == G4_CTAS) ntn = g4_ntn(n16);                           // cluster tiles per row of tiles
    else ntn = (n16 + e.tile_n - 1) / e.tile_n;
    const int nset = (int)(e.sv.uset_ptr[a + 1] - e.sv.uset_ptr[a]);
    int m0 = (int)e.sv.unit_ptr[a];
    const int m1 = (int)e.sv.unit_ptr[a + 1];
    while (m0 + 1 < m1 && (e.sv.unit_mem[m0] < e.atom_lo || e.sv.unit_mem[m0] >= e.atom_hi)) ++m0;   // the feed holds units with a member in range
    const int atom = e.sv.unit_mem[m0];
    __stcg(reinterpret_cast<int4*>(&s->atom), make_int4(atom, n, n16, e.upos[atom]));
    __stcg(reinterpret_cast<int4*>(&s->nbi), make_int4(e.at.nb[atom], ntm, ntn, nset));
    __stcg(reinterpret_cast<int4*>(&s->inv_iters), make_int4(0, 0, 0, 0));            // inv, sign, conv, xcur
    __stcg(reinterpret_cast<int4*>(&s->ycur), make_int4(2, 0, 0, 0));                 // ycur, status, gemm_count, tiles_done
    __stcg(reinterpret_cast<float4*>(&s->res_acc), make_float4(0.f, 1e30f, 0.f, 0.f)); // res_acc, res_prev, res_last, rho_s
    __stcg(reinterpret_cast<float4*>(&s->rho_a), make_float4(0.f, 1.f, 0.5f, 0.f));    // rho_a, alpha1, alpha2, side_done
    __stcg(reinterpret_cast<int4*>(&s->noboost), make_int4(0, a, m0, m1));
    __stcg(&s->resume, 0);
    p_install_side(e, slot, SK_GATHER, (nset + e.gather_rowatoms - 1) / e.gather_rowatoms);
    return true;
}

// Phase FIN finished (or skipped for a failed inverse): publish the atom's results, free / refill the slot.
__device__ __forceinline__ void p_retire(const PEngine& e, int slot) {
    PSlot* s = &e.slots[slot];
    const int a = __ldcg(&s->unit);
    e.at.inv[a] = __ldcg(&s->inv_iters); e.at.sign[a] = __ldcg(&s->sign_iters); e.at.status[a] = __ldcg(&s->status);
    e.at.gemms[a] = __ldcg(&s->gemm_count); e.at.res[a] = __ldcg(&s->res_last); e.at.rho[a] = __ldcg(&s->rho_a);
    const bool more = p_refill(e, slot);
    if (!more) *(volatile unsigned int*)&e.sclaim[slot] = 0u;
    __threadfence();
    atomicAdd(e.finished, 1);
}

// ------------------------------------------------------------------------------------------------
// GEMM side: called by one thread per CTA per finished tile (after the CTA's stores and residual
// atomics). The last report of the op runs the slot's transition (same rules as tile_finished of the
// round engine: DESIGN.md C-7) and installs what comes next.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void p_tile_finished(const PEngine& e, int slot, int nreports) {
    PSlot* s = &e.slots[slot];
    __threadfence();
    const int prev = atomicAdd(&s->tiles_done, 1);
    if (prev != nreports - 1) return;
    __threadfence();
    __stcg(&s->tiles_done, 0);
    const int kind = __ldcg(&s->op_kind);
    if (kind == OP_POW_S || kind == OP_POW_A) {
        // ||alpha M V_k||_F^2 from the fused reduction; rho estimate = growth of the Frobenius norm
        const float r_new = atomicExch(&s->res_acc, 0.0f);
        const float alpha = __ldcg(&s->pow_alpha);
        float est = sqrtf(r_new / __ldcg(&s->pow_norm2)) / alpha;
        if (!(est > 1e-20f) || !(est < 1e20f)) est = 1.f;
        const int step = __ldcg(&s->pow_step) + 1;
        const int P = kind == OP_POW_S ? e.p_s : e.p_a;
        if (step < P) {
            __stcg(&s->pow_step, step);
            __stcg(&s->pow_norm2, r_new);
            __stcg(&s->pow_alpha, 1.f / est);                         // keeps ||V_k||_F at its starting magnitude
            p_install_gemm(e, slot, kind);
        } else if (kind == OP_POW_S) {
            __stcg(&s->rho_s, e.safety_s * est);
            p_install_side(e, slot, SK_SCHULZ1, e.schulz_chunks);
        } else {
            const float rho = e.safety_a * est;
            __stcg(&s->rho_a, rho);
            __stcg(&s->alpha1, 1.f / (rho * rho));
            __stcg(&s->alpha2, 0.5f / rho);
            if (e.split_tokens) { __stcg(&s->resume, 1); p_enter_heavy(e, slot); }
            else p_install_gemm(e, slot, OP_SIGN_G1);
        }
        return;
    }
    if (kind == OP_DCOLS) {                 // a skinny product, not one of the counted square GEMMs
        if (__ldcg(&s->resume) != 2) { __stcg(&s->resume, 2); p_leave_heavy(e, slot); }          // first member served: the chain is over
        p_install_side(e, slot, SK_DCOLS, e.dcols_chunks);
        return;
    }
    __stcg(&s->gemm_count, __ldcg(&s->gemm_count) + 1);
    if (kind == OP_INV_G1 || kind == OP_SIGN_G1) {
        const bool inv = kind == OP_INV_G1;
        const float sum = atomicExch(&s->res_acc, 0.0f);
        const float r = sqrtf(sum / (float)__ldcg(&s->n));
        const float rp = __ldcg(&s->res_prev);
        __stcg(&s->res_prev, r);
        __stcg(&s->res_last, r);
        const float tol = inv ? e.tol_inv : e.tol_sign;
        const int iters = inv ? __ldcg(&s->inv_iters) : __ldcg(&s->sign_iters);
        const int cap = inv ? e.max_inv : e.max_sign;
        const bool ok = r < tol;
        const bool stagnated = (r > 0.5f * rp) && (r < 4.f * tol) && iters > 0;   // rounding floor reached
        // during the scaled sign steps the bulk of the spectrum is deliberately kept away from +-1, so the
        // residual need not fall from one step to the next: the divergence rule applies after them
        const bool scaled_phase = !inv && iters <= e.n_sched && !__ldcg(&s->noboost);
        const bool diverged = !(r == r) || (!scaled_phase && iters > 1 && r > rp && r > 0.9f);
        const bool capped = iters + 1 >= cap;
        if (diverged || (capped && !ok && !stagnated)) __stcg(&s->status, __ldcg(&s->status) | (inv ? ST_NOTSPD : ST_NOCONV));
        const bool conv = ok || stagnated || diverged || capped;
        if (!inv && conv && p_sign_alpha(e, s, iters) != 1.f) {
            // X_k passed the test, but T was formed with alpha_k != 1 and a scaled step would move the spectrum
            // away from +-1 again: switch the scaling off for this matrix and form T = 3I - X_k^2 once more
            __stcg(&s->noboost, 1);
            __stcg(&s->res_prev, rp);
            p_install_gemm(e, slot, OP_SIGN_G1);
            return;
        }
        __stcg(&s->conv, conv ? 1 : 0);
        p_install_gemm(e, slot, inv ? OP_INV_G2 : OP_SIGN_G2);
    } else if (kind == OP_INV_G2) {
        __stcg(&s->inv_iters, __ldcg(&s->inv_iters) + 1);
        __stcg(&s->ycur, 5 - __ldcg(&s->ycur));
        if (__ldcg(&s->conv)) {
            __stcg(&s->conv, 0);
            __stcg(&s->res_prev, 1e30f);
            if (__ldcg(&s->status) & ST_NOTSPD) { p_leave_heavy(e, slot); p_retire(e, slot); }   // no D for this atom (rows stay zero)
            else p_install_gemm(e, slot, OP_AMAT);
        } else {
            p_install_gemm(e, slot, OP_INV_G1);
        }
    } else if (kind == OP_AMAT) {
        if (e.split_tokens) p_leave_heavy(e, slot);              // the token is not held across the power iteration
        p_start_power(e, slot, OP_POW_A);
    } else if (kind == OP_SIGN_G2) {
        __stcg(&s->sign_iters, __ldcg(&s->sign_iters) + 1);
        __stcg(&s->xcur, 1 - __ldcg(&s->xcur));
        if (__ldcg(&s->conv)) {
            __stcg(&s->conv, 0);
            p_install_gemm(e, slot, OP_DCOLS);
        } else {
            p_install_gemm(e, slot, OP_SIGN_G1);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Tile scheduler of the persistent engine (leader CTA, one warp): claims tiles from gclaim[] in slot
// order and publishes them to both CTAs of the pair.
// ------------------------------------------------------------------------------------------------
template <int CTAS>
__device__ __forceinline__ void p_scheduler(const G2Smem& sm, const PEngine& e, int lane) {
    int q = 0; uint32_t ph = 0;
    unsigned long long idle_ns = 0, ntiles = 0, overshoot = 0;
    const unsigned long long t_begin = pl::gtime();
    const int my_die = p_my_die(e);
    for (;;) {
        for (uint32_t spins = 0; !ptx::mbar_try_wait_cluster(sm.ti_empty(q), ph ^ 1);) {
            __nanosleep(100);
            if (++spins > (1u << 26)) __trap();
        }
        // Claim lazily: only when the producer has issued every load of the tile before and needs the next
        // record (it runs G2_STAGES k-blocks ahead of the MMA, which hides the claim). A pair that claimed
        // further ahead would hoard tiles of a GEMM that idle pairs could run at the same time, and the
        // slot's chain of dependent GEMMs would take that much longer.
        for (uint32_t spins = 0; !ptx::mbar_try_wait(sm.want(), (uint32_t)(ntiles & 1) ^ 1u);) {
            __nanosleep(64);
            if (++spins > (1u << 28)) __trap();
        }
        TileInfo ti{};
        int got = 0, half_height = 0;
        unsigned long long t_idle0 = 0;
        for (;;) {
            int found = -1;
            for (int base = 0; base < e.S; base += 32) {
                const int sidx = base + lane;
                const unsigned long long w = sidx < e.S ? *(volatile unsigned long long*)&e.gclaim[sidx] : 0ull;
                const bool avail = (unsigned)(w & 0xFFFFFu) < (unsigned)((w >> 20) & 0xFFFFFu) && (my_die < 0 || (sidx & 1) == my_die);
                const unsigned m = __ballot_sync(0xffffffffu, avail);
                if (m) { found = base + __ffs(m) - 1; break; }
            }
            if (found >= 0) {
                unsigned long long w = 0;
                if (lane == 0) w = atomicAdd(&e.gclaim[found], 1ull);
                w = __shfl_sync(0xffffffffu, w, 0);
                const int t = (int)(w & 0xFFFFFu), nt = (int)((w >> 20) & 0xFFFFFu);
                if (t < nt) {
                    if (lane == 0) {
                        __threadfence();
                        const PSlot* s = &e.slots[found];
                        const int4 g0 = __ldcg(reinterpret_cast<const int4*>(&s->atom));     // atom n n16 pos
                        const int4 g1 = __ldcg(reinterpret_cast<const int4*>(&s->nbi));      // nbi ntm ntn nset
                        const int4 o0 = __ldcg(reinterpret_cast<const int4*>(&s->op_kind));
                        const float4 o1 = __ldcg(reinterpret_cast<const float4*>(&s->c_out));
                        const bool pow = o0.x == OP_POW_S || o0.x == OP_POW_A || o0.x == OP_DCOLS;
                        const int ntn = pow ? 1 : g1.z;
                        const int tm = t / ntn, tn = t - tm * ntn;
                        ti.slot = found; ti.m0 = tm * BM;
                        if (o0.x == OP_DCOLS) { ti.n0 = g0.w & ~7; ti.bn = PCW; }          // D columns: the aligned window around pos(i), pair 0 only
                        else if (pow) { ti.n0 = 0; ti.bn = NVC; }                          // pair 0 only
                        else if (CTAS == G4_CTAS) {
                            int n0, bn0, bn1;
                            g4_cols(g0.z, tn, n0, bn0, bn1);
                            ti.n0 = n0; ti.bn = bn0 | (bn1 << 16);
                        } else {
                            ti.n0 = tn * e.tile_n; ti.bn = min(e.tile_n, g0.z - tn * e.tile_n);
                            // the last row block when at most 128 rows are left: one M = 128 MMA per 16 k instead of M = 256
                            if (e.half_tiles && g0.z - tm * BM <= BM / 2 && (ti.bn & 31) == 0) half_height = 1;
                        }
                        ti.n = g0.y; ti.n16 = g0.z; ti.nreports = CTAS * nt;
                        ti.kind = o0.x; ti.a_buf = o0.y; ti.b_buf = o0.z; ti.c_buf = o0.w;
                        ti.c_out = o1.x; ti.alpha_res = o1.y; ti.beta = o1.z; ti.want_res = __float_as_int(o1.w);
                    }
                    got = 1;
                    break;
                }
                ++overshoot;
                continue;
            }
            if (*(volatile int*)e.finished >= e.total || *e.abort_flag) break;
            if (!t_idle0) t_idle0 = pl::gtime();
            __nanosleep(200);
        }
        if (t_idle0) idle_ns += pl::gtime() - t_idle0;
        ntiles += got;
        if (lane == 0) ti.valid = got ? (1 | (half_height << 1)) : 0;
        const uint32_t* w = reinterpret_cast<const uint32_t*>(&ti);
        uint32_t mine = 0;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const uint32_t v = __shfl_sync(0xffffffffu, w[i], 0);
            if (lane == i) mine = v;
        }
        if (lane < 16) {
#pragma unroll
            for (uint32_t rk = 0; rk < (uint32_t)CTAS; ++rk)
                ptx::st_cluster_u32(ptx::mapa(sm.tinfo(q), rk) + 4u * lane, mine);
        }
        __syncwarp();
        if (lane < CTAS) ptx::mbar_arrive_cluster(ptx::mapa(sm.ti_full(q), (uint32_t)lane));
        if (!got) break;
        if (++q == G2_NTI) { q = 0; ph ^= 1; }
    }
    if (lane == 0) {
        const unsigned long long t_end = pl::gtime();
        atomicAdd(&e.ctr[PC_TILES], ntiles);
        atomicAdd(&e.ctr[PC_SCHED_IDLE_NS], idle_ns);
        atomicAdd(&e.ctr[PC_SCHED_BUSY_NS], t_end - t_begin - idle_ns);
        atomicAdd(&e.ctr[PC_OVERSHOOT], overshoot);
        atomicMin(&e.ctr[PC_T_START], t_begin);
        atomicMax(&e.ctr[PC_T_END], t_end);
    }
}

// ================================================================================================
// Side tasks. `tid` in [0, P_SIDE_THREADS); `sm` is the side group's shared memory (P_SIDE_SMEM bytes).
// One side group is four warps on an SM that is busy with GEMM tiles, so every loop is written for
// memory-level parallelism: several independent loads are issued before the first one is used.
// ================================================================================================

// a1, one chunk of row-atoms of the unit's index set N (N(i), or the union over the unit's members): builds the dense
// rows of T(S) (buffer 0) and T(H0) (buffer 1) that belong to row-atoms [a_lo, a_hi) of N: block (j_a, j_b) of the sparse matrix where it exists,
// zeros elsewhere and in the pad strip [n, n16). The last chunk also zeroes rows [n, n16).
//
// Data path: the source blocks of a row-atom are contiguous runs of nb(j_a) x nb(j_b) values. All of them (S and H0) are
// prefetched into L2 first; every warp then loads G_NB blocks at a time with coalesced 8-byte loads, converts each value
// once (RN-even, C-13) into a shared-memory strip of the dense rows, and the strip leaves with 16-byte
// coalesced stores. Strips are G_STRIP_BYTES at most, so a row-atom of a very wide submatrix takes several passes over
// row sub-ranges of its blocks.
constexpr int G_STRIP_BYTES = 48 * 1024;
constexpr int G_NB = 2;                           // blocks a warp has in flight (8 loads per lane each)

template <typename TV>
__device__ void side_gather_chunk(const SysView& sv, const TV* __restrict__ S_vals, const TV* __restrict__ H_vals,
                                  __half* __restrict__ dstS, __half* __restrict__ dstH, int unit, int n, int n16, int ld,
                                  int chunk, int nchunks, unsigned char* sm, int tid, unsigned long long* bytes, int e_prefetch = 1) {
    const long long p0 = sv.uset_ptr[unit];
    const int cnt = (int)(sv.uset_ptr[unit + 1] - p0);
    const int warp = tid >> 5, lane = tid & 31;
    // shared memory: tables | strip
    int* s_nset = reinterpret_cast<int*>(sm);                              // [cnt] atoms of N(i)
    int* s_off = s_nset + cnt;                                             // [cnt + 1] first column of each atom
    int* s_list = s_off + cnt + 1;                                         // [cnt] present blocks of the current row-atom
    int* s_m = s_list + cnt;                                               // [1]
    long long* s_boff = reinterpret_cast<long long*>(sm + (((size_t)(3 * cnt + 2) * 4 + 15) & ~(size_t)15));   // [cnt]
    unsigned char* strip_b = reinterpret_cast<unsigned char*>(s_boff) + (((size_t)cnt * 8 + 15) & ~(size_t)15);
    __half* strip = reinterpret_cast<__half*>(strip_b);

    const int a_lo = (int)((long long)cnt * chunk / nchunks), a_hi = (int)((long long)cnt * (chunk + 1) / nchunks);
    for (int b = tid; b < cnt; b += P_SIDE_THREADS) { s_nset[b] = sv.uset_atom[p0 + b]; s_off[b] = sv.uset_off[p0 + b]; }
    if (tid == 0) s_off[cnt] = n;
    pl::side_sync();
    const int rows_max = max(1, G_STRIP_BYTES / (n16 * 2));
    const int vpr = n16 >> 3;                                              // 16-byte vectors per dense row
    unsigned long long nread = 0;

#ifdef NOLSM_TIMING
    long long tp_[4] = {0, 0, 0, 0}, tq_ = clock64();
#define GT_(i) do { const long long t_ = clock64(); tp_[i] += t_ - tq_; tq_ = t_; } while (0)
#else
#define GT_(i)
#endif
    for (int a = a_lo; a < a_hi; ++a) {
        const int j = s_nset[a];
        const int nbj = s_off[a + 1] - s_off[a], row0 = s_off[a];
        // CSR row of j against N(i) (both ascending): every entry looks itself up in N(i)
        for (int b = tid; b < cnt; b += P_SIDE_THREADS) s_boff[b] = -1;
        pl::side_sync();
        {
            const long long r0 = sv.row_ptr[j], r1 = sv.row_ptr[j + 1];
            for (long long p = r0 + tid; p < r1; p += P_SIDE_THREADS) {
                const int k = sv.col_idx[p];
                int lo = 0, hi = cnt;
                while (lo < hi) { const int mid = (lo + hi) >> 1; if (s_nset[mid] < k) lo = mid + 1; else hi = mid; }
                if (lo < cnt && s_nset[lo] == k) s_boff[lo] = sv.blk_off[p];
            }
        }
        pl::side_sync();
        if (warp == 0) {                                                   // compact list of the present blocks
            int m = 0;
            for (int base = 0; base < cnt; base += 32) {
                const int b = base + lane;
                const bool pr = b < cnt && s_boff[b] >= 0;
                const unsigned mask = __ballot_sync(0xffffffffu, pr);
                if (pr) s_list[m + __popc(mask & ((1u << lane) - 1u))] = b;
                m += __popc(mask);
            }
            if (lane == 0) *s_m = m;
        }
        pl::side_sync();
        const int m = *s_m;
        // L2 prefetch of every source block of this row-atom (S and H0): the staged loads below can keep only ~24 KB in
        // flight per side group, a prefetch needs no shared memory, so all but the first stage round find their lines in L2
        if (e_prefetch) {
            const int nbmax = s_off[cnt] > 0 ? 32 : 32;            // lines per block: computed per block below
            (void)nbmax;
            for (int q = tid; q < m; q += P_SIDE_THREADS) {
                const int b = s_list[q];
                const long long bo = s_boff[b];
                const int bytes_b = nbj * (s_off[b + 1] - s_off[b]) * (int)sizeof(TV);
                const char* ps = reinterpret_cast<const char*>(S_vals + bo);
                const char* ph = reinterpret_cast<const char*>(H_vals + bo);
                for (int o = 0; o < bytes_b + 127; o += 128) {
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(ps + min(o, bytes_b - 1)));
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(ph + min(o, bytes_b - 1)));
                }
            }
        }
        GT_(0);
#pragma unroll 1
        for (int which = 0; which < 2; ++which) {
            const TV* __restrict__ vals = which ? H_vals : S_vals;
            __half* __restrict__ dst = which ? dstH : dstS;
#pragma unroll 1
            for (int r0 = 0; r0 < nbj; r0 += rows_max) {
                const int nr = min(rows_max, nbj - r0);
                {   // zero the strip
                    const uint4 z = make_uint4(0, 0, 0, 0);
                    uint4* s4 = reinterpret_cast<uint4*>(strip);
                    for (int q = tid; q < nr * vpr; q += P_SIDE_THREADS) s4[q] = z;
                }
                pl::side_sync();
                GT_(1);
                // ---- each warp takes G_NB blocks at a time: all their loads are issued (coalesced 8-byte loads, G_NB x 8 per
                //      lane in flight) before the first value is converted into the strip. (8-byte cp.async staging ran at
                //      ~8 cycles per element in the load/store unit and made the gather the busiest side task.) ----
#pragma unroll 1
                for (int l0 = warp * G_NB; l0 < m; l0 += P_SIDE_WARPS * G_NB) {
                    TV v[G_NB][8];
#pragma unroll
                    for (int u = 0; u < G_NB; ++u) {
                        const int li = l0 + u;
                        if (li < m) {
                            const int b = s_list[li];
                            const int nbb = s_off[b + 1] - s_off[b], bs = nr * nbb;
                            const TV* src = vals + s_boff[b] + (long long)r0 * nbb;
#pragma unroll
                            for (int k = 0; k < 8; ++k) {
                                const int e = lane + 32 * k;
                                v[u][k] = e < bs ? __ldg(src + e) : (TV)0;
                            }
                            nread += (lane == 0) ? (unsigned long long)bs : 0ull;
                        }
                    }
#pragma unroll
                    for (int u = 0; u < G_NB; ++u) {
                        const int li = l0 + u;
                        if (li < m) {
                            const int b = s_list[li];
                            const int nbb = s_off[b + 1] - s_off[b], bs = nr * nbb, c0 = s_off[b];
#pragma unroll
                            for (int k = 0; k < 8; ++k) {
                                const int e = lane + 32 * k;
                                if (e < bs) {
                                    const int rr = e / nbb, cc = e - rr * nbb;
                                    strip[rr * n16 + c0 + cc] = Num<__half>::from_d((double)v[u][k]);
                                }
                            }
                        }
                    }
                }
                pl::side_sync();
                GT_(2);
                // ---- the strip leaves with 16-byte stores ----
                {
                    const uint4* s4 = reinterpret_cast<const uint4*>(strip);
                    for (int q = tid; q < nr * vpr; q += P_SIDE_THREADS) {
                        const int rr = q / vpr, v = q - rr * vpr;
                        *reinterpret_cast<uint4*>(dst + (long long)(row0 + r0 + rr) * ld + v * 8) = s4[q];
                    }
                }
                pl::side_sync();
                GT_(3);
            }
        }
    }
#ifdef NOLSM_TIMING
    if (tid == 0) for (int i_ = 0; i_ < 4; ++i_) atomicAdd(&g4_timing[12 + i_], (unsigned long long)tp_[i_]);
#endif
    if (chunk == nchunks - 1) {
        const uint4 z = make_uint4(0, 0, 0, 0);
        for (int idx = tid; idx < (n16 - n) * vpr; idx += P_SIDE_THREADS) {
            const int rr = idx / vpr, v = idx - rr * vpr;
            *reinterpret_cast<uint4*>(dstS + (long long)(n + rr) * ld + v * 8) = z;
            *reinterpret_cast<uint4*>(dstH + (long long)(n + rr) * ld + v * 8) = z;
        }
    }
    if (bytes) {
        if (lane == 0 && nread) atomicAdd(bytes, nread * sizeof(TV));                                  // source values read
        if (tid == 0) atomicAdd(bytes, (unsigned long long)(s_off[a_hi] - s_off[a_lo]) * n16 * 4ull); // dense FP16 rows written (S and H0)
    }
}

// First Schulz step in closed form, rows [r_lo, r_hi) of n16: Y1 = (2/rho) I - S / rho^2 inside
// [0, n)^2, zero in the pad strip (C-8).
__device__ void side_schulz1_chunk(const __half* __restrict__ S, __half* __restrict__ Y, int n, int n16, int ld, float rho,
                                   int chunk, int nchunks, int tid) {
    const int r_lo = (int)((long long)n16 * chunk / nchunks), r_hi = (int)((long long)n16 * (chunk + 1) / nchunks);
    const float d = 2.f / rho, sc = 1.f / (rho * rho);
    const int ppr = n16 >> 3;
    const int total = (r_hi - r_lo) * ppr;
    constexpr int U = 8;
#pragma unroll 1
    for (int idx0 = tid; idx0 < total; idx0 += U * P_SIDE_THREADS) {
        uint4 u[U];
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int idx = idx0 + q * P_SIDE_THREADS;
            if (idx < total) {
                const int rl = idx / ppr, p = idx - rl * ppr;
                u[q] = __ldcg(reinterpret_cast<const uint4*>(S + (long long)(r_lo + rl) * ld + p * 8));
            }
        }
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int idx = idx0 + q * P_SIDE_THREADS;
            if (idx < total) {
                const int rl = idx / ppr, p = idx - rl * ppr;
                const int r = r_lo + rl, c0 = p * 8;
                const __half2* h = reinterpret_cast<const __half2*>(&u[q]);
                float f[8];
#pragma unroll
                for (int w = 0; w < 4; ++w) { const float2 t = __half22float2(h[w]); f[2 * w] = t.x; f[2 * w + 1] = t.y; }
#pragma unroll
                for (int w = 0; w < 8; ++w) {
                    const int c = c0 + w;
                    f[w] = (r < n && c < n) ? ((r == c ? d : 0.f) - sc * f[w]) : 0.f;
                }
                st_half8(Y + (long long)r * ld + c0, f);
            }
        }
    }
}

// a6 + a7, one chunk of the values of output row i (slot (i, j) holds (D_ji)^T, C-10):
// D_sub[r, pos + c] = 1/2 (Y[r, pos + c] - P[r, c]) with P = X Y[:, cols(i)] from the OP_DCOLS tiles, and the
// energy partial sum <D_ji, H0_ji> in FP64 (Eq. 4). One thread per output value, in output
// order: the block-CSR arrays (D out, H0 in) are touched with coalesced accesses, the small L2-resident
// operands (Y columns, P) with scattered ones.
template <typename TV, typename TD>
__device__ void side_dcols_chunk(const SysView& sv, const float* __restrict__ P, const __half* __restrict__ Y,
                                 const TV* __restrict__ H_vals, const TV* __restrict__ S_vals, TD* __restrict__ D_vals, double* e_atom,
                                 double* q_atom, int atom, int n_own, int ld, int pos, int nbi, int chunk, int nchunks, unsigned char* sm, int tid) {
    const long long p0 = sv.nset_ptr[atom];
    const int cnt = (int)(sv.nset_ptr[atom + 1] - p0);
    int* s_pre = reinterpret_cast<int*>(sm);                               // [cnt + 1] first value row of each atom of N(i) in output order
    int* s_row = s_pre + cnt + 1;                                          // [cnt] first row of that atom inside the unit's matrix
    for (int b = tid; b < cnt; b += P_SIDE_THREADS) { s_pre[b] = sv.nset_off[p0 + b]; s_row[b] = sv.nset_uoff[p0 + b]; }
    if (tid == 0) s_pre[cnt] = n_own;
    pl::side_sync();
    // value q of the chunk = (atom a of N(i), column c, row bb) in output order; the rows of atom a sit at s_row[a]
    // of the unit's matrix (== s_pre[a] when the unit is the atom itself)
    const int total = n_own * nbi;                                         // values of D written for this atom
    const int q_lo = (int)((long long)total * chunk / nchunks), q_hi = (int)((long long)total * (chunk + 1) / nchunks);
    double e_part = 0.0, q_part = 0.0;
    for (int q = q_lo + tid; q < q_hi; q += P_SIDE_THREADS) {
        int lo = 0, hi = cnt - 1;
        while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (s_pre[mid] * nbi <= q) lo = mid; else hi = mid - 1; }
        const int a = lo, nbj = s_pre[a + 1] - s_pre[a];
        const int rem = q - s_pre[a] * nbi;
        const int c = rem / nbj, bb = rem - c * nbj;
        const int r = s_row[a] + bb;
        const long long o = sv.blk_off[sv.nset_slot[p0 + a]] + rem;       // slot (i, j_a): [c][bb] = D_sub[r, pos + c]
        const float d = 0.5f * (__half2float(__ldcg(Y + (long long)r * ld + pos + c)) - __ldcg(P + (size_t)r * PCW + (pos & 7) + c));
        D_vals[o] = (TD)d;
        e_part += (double)d * (double)H_vals[o];
        q_part += (double)d * (double)S_vals[o];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { e_part += __shfl_xor_sync(0xffffffffu, e_part, o); q_part += __shfl_xor_sync(0xffffffffu, q_part, o); }
    if ((tid & 31) == 0 && e_part != 0.0) atomicAdd(&e_atom[atom], e_part);
    if ((tid & 31) == 0 && q_part != 0.0) atomicAdd(&q_atom[atom], q_part);
}

// ------------------------------------------------------------------------------------------------
// Side group main loop.
// ------------------------------------------------------------------------------------------------
__device__ void p_side_loop(const PEngine& e, unsigned char* sm, int tid) {
    __shared__ int s_ctl[4];                      // slot, kind, chunk, nchunks
    const int warp = tid >> 5, lane = tid & 31;
    const int my_die = p_my_die(e);
    unsigned long long busy_ns[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tasks[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (;;) {
        if (warp == 0) {
            int slot = -1, kind = -1, chunk = 0, nch = 0;
            for (;;) {
                int found = -1;
                for (int base = 0; base < e.S; base += 32) {
                    const int sidx = base + lane;
                    const unsigned w = sidx < e.S ? *(volatile unsigned int*)&e.sclaim[sidx] : 0u;
                    const bool avail = (w & 0x3FFFu) < ((w >> 14) & 0x3FFFu) && (my_die < 0 || (sidx & 1) == my_die);
                    const unsigned m = __ballot_sync(0xffffffffu, avail);
                    if (m) { found = base + __ffs(m) - 1; break; }
                }
                if (found >= 0) {
                    unsigned w = 0;
                    if (lane == 0) w = atomicAdd(&e.sclaim[found], 1u);
                    w = __shfl_sync(0xffffffffu, w, 0);
                    const int c = (int)(w & 0x3FFFu), n = (int)((w >> 14) & 0x3FFFu);
                    if (c < n) { slot = found; kind = (int)(w >> 28); chunk = c; nch = n; break; }
                    continue;
                }
                if (*(volatile int*)e.finished >= e.total || *e.abort_flag) break;
                __nanosleep(500);
            }
            if (lane == 0) { s_ctl[0] = slot; s_ctl[1] = kind; s_ctl[2] = chunk; s_ctl[3] = nch; }
        }
        pl::side_sync();
        const int slot = s_ctl[0], kind = s_ctl[1], chunk = s_ctl[2], nch = s_ctl[3];
        if (kind < 0) break;
        __threadfence();
        const unsigned long long t0 = pl::gtime();
        PSlot* s = &e.slots[slot];
        const int4 g0 = __ldcg(reinterpret_cast<const int4*>(&s->atom));     // atom n n16 pos
        const int4 g1 = __ldcg(reinterpret_cast<const int4*>(&s->nbi));      // nbi ntm ntn nset
        const int atom = g0.x, n = g0.y, n16 = g0.z, pos = g0.w, nbi = g1.x;
        switch (kind) {
            case SK_GATHER: {
                __half* dS = e.base + buf_off(e, slot, 0);
                __half* dH = e.base + buf_off(e, slot, 1);
                if (e.val_f64) side_gather_chunk<double>(e.sv, (const double*)e.S_vals, (const double*)e.H_vals, dS, dH, __ldcg(&s->unit), n, n16, e.ld, chunk, nch, sm, tid, &e.ctr[PC_SIDE_BYTES + SK_GATHER], e.gather_prefetch);
                else side_gather_chunk<float>(e.sv, (const float*)e.S_vals, (const float*)e.H_vals, dS, dH, __ldcg(&s->unit), n, n16, e.ld, chunk, nch, sm, tid, &e.ctr[PC_SIDE_BYTES + SK_GATHER], e.gather_prefetch);
            } break;
            case SK_SCHULZ1:
                side_schulz1_chunk(e.base + buf_off(e, slot, 0), e.base + buf_off(e, slot, 2), n, n16, e.ld, __ldcg(&s->rho_s), chunk, nch, tid);
                break;
            case SK_DCOLS: {
                const float* P = pcols_ptr(e, slot);
                const __half* Y = e.base + buf_off(e, slot, __ldcg(&s->ycur));
                if (e.val_f64) {
                    if (e.d_f64) side_dcols_chunk<double, double>(e.sv, P, Y, (const double*)e.H_vals, (const double*)e.S_vals, (double*)e.D_vals, e.e_atom, e.q_atom, atom, e.adim[atom], e.ld, pos, nbi, chunk, nch, sm, tid);
                    else side_dcols_chunk<double, float>(e.sv, P, Y, (const double*)e.H_vals, (const double*)e.S_vals, (float*)e.D_vals, e.e_atom, e.q_atom, atom, e.adim[atom], e.ld, pos, nbi, chunk, nch, sm, tid);
                } else {
                    if (e.d_f64) side_dcols_chunk<float, double>(e.sv, P, Y, (const float*)e.H_vals, (const float*)e.S_vals, (double*)e.D_vals, e.e_atom, e.q_atom, atom, e.adim[atom], e.ld, pos, nbi, chunk, nch, sm, tid);
                    else side_dcols_chunk<float, float>(e.sv, P, Y, (const float*)e.H_vals, (const float*)e.S_vals, (float*)e.D_vals, e.e_atom, e.q_atom, atom, e.adim[atom], e.ld, pos, nbi, chunk, nch, sm, tid);
                }
            } break;
            default: break;                       // SK_REFILL: nothing to compute
        }
        ptx::fence_proxy_async();                 // buffers written here are read next by TMA
        pl::side_sync();
        if (tid == 0) {
            busy_ns[kind & 7] += pl::gtime() - t0;
            tasks[kind & 7] += 1;
            __threadfence();
            const int prev = nch > 1 ? atomicAdd(&s->side_done, 1) : 0;
            if (prev == nch - 1) {
                __threadfence();
                if (nch > 1) __stcg(&s->side_done, 0);
                switch (kind) {
                    case SK_REFILL:
                        if (!p_refill(e, slot)) *(volatile unsigned int*)&e.sclaim[slot] = 0u;
                        break;
                    case SK_GATHER: p_start_power(e, slot, OP_POW_S); break;
                    case SK_SCHULZ1: p_enter_heavy(e, slot); break;
                    case SK_DCOLS: {
                        const double nv = (double)(e.sv.blk_off[e.sv.row_ptr[atom + 1]] - e.sv.blk_off[e.sv.row_ptr[atom]]);
                        atomicAdd(&e.ctr[PC_SIDE_BYTES + SK_DCOLS],
                                  (unsigned long long)(nv * ((e.d_f64 ? 8 : 4) + (e.val_f64 ? 8 : 4)) + (double)n * PCW * 4.0 + (double)n * nbi * 2.0));
                        // the next member of the unit takes its columns from the same X and Y, or the slot retires
                        int mp = __ldcg(&s->mptr) + 1;
                        const int mend = __ldcg(&s->mend);
                        while (mp < mend && (e.sv.unit_mem[mp] < e.atom_lo || e.sv.unit_mem[mp] >= e.atom_hi)) ++mp;
                        if (mp < mend) {
                            const int nxt = e.sv.unit_mem[mp];
                            __stcg(&s->mptr, mp);
                            __stcg(&s->atom, nxt);
                            __stcg(&s->pos, e.upos[nxt]);
                            __stcg(&s->nbi, e.at.nb[nxt]);
                            p_install_gemm(e, slot, OP_DCOLS);
                        } else {
                            p_retire(e, slot);
                        }
                    } break;
                    default: break;
                }
            }
        }
    }
    if (tid == 0)
        for (int k = 0; k < 8; ++k) {
            if (busy_ns[k]) atomicAdd(&e.ctr[PC_SIDE_NS + k], busy_ns[k]);
            if (tasks[k]) atomicAdd(&e.ctr[PC_SIDE_TASKS + k], tasks[k]);
        }
}

// ================================================================================================
// The kernel.
// ================================================================================================
// CTAS = CTAs per cluster (set at launch): 2 = pair tiles (gemm2sm.cuh), 4 = two pairs sharing A (gemm4sm.cuh).
template <int CTAS>
__global__ void __launch_bounds__(P_THREADS, 1)
nolsm_persist_kernel(const __grid_constant__ PEngine e) {
    extern __shared__ uint8_t smem_raw[];
    G2Smem sm;
    sm.base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* side_sm = smem_raw + (sm.base - ptx::smem_u32(smem_raw)) + (G2_SMEM_BYTES - 1024);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();
    auto done = [&](const TileInfo& ti) { p_tile_finished(e, ti.slot, ti.nreports); };

    uint32_t tmem_base;
    if constexpr (CTAS == G4_CTAS) tmem_base = g4_setup(sm, warp, lane);
    else tmem_base = g2_setup(sm, warp, lane);

    if (warp < G2_EPI_WARPS) {
        if constexpr (CTAS == G4_CTAS) g4_epilogue(sm, tmem_base, e, e.base, rank, warp, lane, done);
        else g2_epilogue(sm, tmem_base, e, e.base, rank, warp, lane, done, e.tma_store ? e.maps : nullptr);
    } else if (warp == G2_WARP_SCHED) {
        if (rank == 0) p_scheduler<CTAS>(sm, e, lane);
    } else if (warp == G2_WARP_TMA) {
        if constexpr (CTAS == G4_CTAS) g4_producer(sm, e.maps, rank, lane, e.want_lead, e.dbg);
        else g2_producer(sm, e.maps, rank, lane, e.want_lead);
    } else if (warp == G2_WARP_MMA) {
        if constexpr (CTAS == G4_CTAS) { if ((rank & 1u) == 0) g4_mma(sm, tmem_base, rank, lane, e.dbg); }
        else { if (rank == 0) g2_mma(sm, tmem_base, lane); }
    } else {
        p_side_loop(e, side_sm, (int)threadIdx.x - G2_CTRL_THREADS);
    }
    g2_teardown(tmem_base, warp);
}

// Stand-alone launch of the gather task for one slot (diagnostics: nolsm_gather_submatrix and the
// HBM-bandwidth measurement of the gather code without the GEMMs). grid = (chunks, slots).
template <typename TV>
__global__ void __launch_bounds__(P_SIDE_THREADS) k_side_gather(SysView sv, const TV* S_vals, const TV* H_vals, __half* base,
                                                                long long slotsz, long long bufsz, int ld, const int* atoms,
                                                                const int* dims, unsigned long long* bytes) {
    extern __shared__ unsigned char sm_dyn[];
    const int atom = atoms[blockIdx.y], n = dims[atom], n16 = (n + 15) & ~15;      // unit id and its dimension
    __half* dS = base + (long long)blockIdx.y * slotsz;
    side_gather_chunk<TV>(sv, S_vals, H_vals, dS, dS + bufsz, atom, n, n16, ld, blockIdx.x, gridDim.x, sm_dyn, threadIdx.x, bytes);
}

}  // namespace nolsm
