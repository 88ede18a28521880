// Persistent engine: the whole hot path a1-a7 of one nolsm_density_matrix call in ONE kernel launch.
//
// grid = one CTA per SM in clusters of two (one tcgen05 CTA pair per tile, gemm2sm.cuh); every CTA runs
//   warps 0-10   the grouped tcgen05 GEMM pipeline of gemm2sm.cuh (epilogue x 8, tile scheduler, TMA
//                producer, MMA issuer in the leader CTA / tile finisher in the peer CTA), fed from a device-side
//                claim table instead of a static tile list;
//   warps 11-14  a SIDE GROUP that executes the O(n^2) steps of the path as small tasks: gather
//                (PAPER.md:L56, L60), the closed-form first iteration steps, diagonal shifts, and D columns +
//                scatter + energy (Eq. 4).
// The spectral scalings (rho(S_sub) for the start of the inverse iteration, rho(A_sub) for X0 = A / rho, C-6)
// come from a BLOCK power iteration with 16 vectors that runs as 256 x 16 GEMM tiles in the same
// pipeline (V <- alpha M V, Frobenius norm of the product from the fused residual reduction).
//
// Two chains of matrix iterations are built on the same machinery (PEngine::lowdin, C-21):
//   0  Eq. 6 as printed: Y = S^-1 by the Schulz iteration, A = Y H0 - mu I, X <- 1/2 X (3I - X^2), D = 1/2 (I - X) Y.
//      S, Y and R = 2I - S Y are polynomials of S: symmetric, so the Schulz GEMMs multiply only the tiles on and above
//      the diagonal (TI_MIRROR, gemm2sm.cuh); A and the sign iterates are not symmetric.
//   1  the symmetric (Loewdin) form, "other iteration schemes that only require scalings, additions and
//      multiplications": Z = S^-1/2 by the coupled Newton-Schulz iteration T = 1/2 (3I - Z Y), Y <- Y T, Z <- T Z,
//      Ht = Z H0 Z - mu I (symmetric), the same Eq. 6 sign iteration on Ht, D = Z 1/2 (I - X) Z. Every iterate is
//      symmetric: all GEMMs but one (H0 Z) multiply the upper triangle of tiles only.
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
// Cross-CTA data flow: GEMM outputs are written with generic stores or TMA stores and read back by TMA (async proxy)
// of other CTAs: writers fence (fence.proxy.async, __threadfence / bulk wait) before the completing atomic; readers
// fence.proxy.async after the claim. Slot state is read and written with .cg accesses (L1 is not
// coherent across SMs).
#pragma once
#include "gemm2sm.cuh"
#include "kernels.cuh"

namespace nolsm {

constexpr int P_SIDE_WARPS = 4;
constexpr int P_SIDE_THREADS = P_SIDE_WARPS * 32;
constexpr int P_THREADS = G2_CTRL_THREADS + P_SIDE_THREADS;
constexpr int P_SIDE_SMEM = 60 * 1024;
constexpr int P_SMEM_BYTES = G2_SMEM_BYTES + P_SIDE_SMEM;
constexpr int P_MAX_CAP = 4096;
constexpr int P_MAX_MU = 8;                     // trial chemical potentials per call (nolsm_electron_counts)

enum SideKind { SK_NONE = 0, SK_REFILL, SK_GATHER, SK_ELEM, SK_DCOLS, SK_WCOLS };
// elementwise side task SK_ELEM: dst = d I - sc src (PSlot::elem_kind says which)
enum ElemKind { EL_SCHULZ1 = 0,   // Y1 = (2/rho) I - S / rho^2                 (first Schulz step, C-8)
                EL_LW1,           // T0 = Z1 = 3/2 I - S / (2 rho)               (first coupled Newton-Schulz step, C-21)
                EL_SHIFT };       // X0 buffer = A0 - mu_j I                     (next trial mu on the resident A0, C-20)

// counters written by the kernel (unsigned long long each)
enum { PC_TILES = 0, PC_SCHED_IDLE_NS, PC_SCHED_BUSY_NS, PC_OVERSHOOT, PC_T_START, PC_T_END,
       PC_SIDE_NS,            // + kind
       PC_SIDE_BYTES = PC_SIDE_NS + 8,   // + kind (algorithmic bytes)
       PC_SIDE_TASKS = PC_SIDE_BYTES + 8,
       PC_MMA_NS = PC_SIDE_TASKS + 8,    // + 0 tile-record wait, 1 accumulator wait, 2 k-loops (MMA warps of the leader CTAs)
       PC_SCHED_RING_NS = PC_MMA_NS + 3, // tile schedulers: waiting for a free ring entry (= for the completion of the tile four back)
       PC_SCHED_CREDIT_NS,               // ... for the producer's claim point
       PC_POW_EXTRA,                     // power-iteration steps for rho(A) beyond p_a (estimate not settled, see p_tile_finished)
       PC_LEN };

constexpr int OPF_RES = 1;        // op flags: fused residual wanted
constexpr int OPF_SYM = 2;        // symmetric product: upper-triangle tiles, mirrored stores
constexpr int OPF_NARROW = 4;     // one narrow tile per row block (power iteration, D columns)

struct __align__(16) PSlot {      // 176 bytes
    int atom, n, n16, pos;                                          // geometry (written at refill; atom / pos / nbi describe member mptr)
    int nbi, ntm, nset, unit;
    int op_kind, a_buf, b_buf, c_buf;                               // live GEMM op: C = c_out A B + beta I, residual of alpha_res A B
    float c_out, alpha_res, beta; int op_flags;
    int inv_iters, sign_iters, conv, xcur;
    int ycur, status, gemm_count, tiles_done;
    float res_acc, res_prev, res_last, rho_s;
    float rho_a, alpha1, alpha2; int side_done;
    int pow_step; float pow_norm2, pow_alpha; int resume;           // block power iteration state; resume: which token phase comes next
    int noboost, mptr, mend, zcur;                                  // noboost: the scaled steps are over for this matrix; members [mptr, mend) still to be served
    int xsum, pow_buf, mu_idx, sym_count;                           // X ping-pong: next = xsum - xcur; buffer of the running power iteration; trial mu; symmetric GEMMs run
    int elem_kind, abuf, op_seq; float pow_g;                       // pow_g: growth est_k / est_{k-1} of the last power step. SK_ELEM variant; buffer that keeps the mu-independent A0 (several trial mu); ops installed so far
};

struct PEngine {
    PSlot* slots;
    unsigned long long* gclaim;   // [S] GEMM claim words
    unsigned int* sclaim;         // [S] side-task claim words
    int S, cap, ld;
    long long bufsz, slotsz;
    float tol_inv, tol_sign, safety_s, safety_a;
    int max_inv, max_sign, p_s, p_a;
    int p_cap;                    // the power iteration for rho(A) may run on up to this many steps while its estimate is not settled
    int gather_rowatoms, elem_chunks, dcols_chunks;   // row-atoms of N(i) per gather chunk; chunks of the other tasks
    int* next_atom; int a_end, total;                 // feed position, its end, units of this call
    const int* feed;              // feed position -> unit id (nullptr: the position is the unit id)
    int atom_lo, atom_hi;         // only members inside [atom_lo, atom_hi) get their columns of D (nolsm_density_matrix_range)
    int* finished;
    int* heavy;                   // [1] slots inside the GEMM-heavy phases right now (at most g_max)
    int* parked;                  // [S] 1 = the slot is ready for a heavy phase and waits for a token
    int g_max, want_lead;
    int scan_rotate;              // 1: pair p scans the claim table from slot 13 p mod S on; 0: every pair from slot 0 (slot-order priority)
    int l2_load, l2_store;        // L2 eviction priority of the operand loads / of the stores of C (1 evict_first, 2 evict_last, 3 normal)
    int lowdin;                   // 0: Eq. 6 on A = S^-1 H0 - mu I; 1: symmetric (Loewdin) form
    int sym_tiles;                // 1: symmetric products multiply the upper triangle of tiles only
    int trans_tiles;              // 1: tiles of a ragged last row block are computed transposed (TI_TRANS)
    int n_mu; float mu[P_MAX_MU]; // trial chemical potentials of this call (1 for nolsm_density_matrix)
    int count_only;               // 1: D is not written, only e and q per trial mu (nolsm_electron_counts)
    double* nelec_mu;             // [P_MAX_MU] sum_i q_i per trial mu (count_only)
    double* e_mu;                 // [P_MAX_MU] sum_i e_i per trial mu (count_only)
    int n_sched; float alpha_sched[16];   // scaled Newton-Schulz: alpha_k of sign iteration k < n_sched (1 afterwards)
    volatile int* abort_flag;     // device word; 1: the host stops a kernel that overran its time limit, 2: a wait stalled (watchdog)
    unsigned long long* ctr;      // [PC_LEN]
    AtomArrays at;                // results are indexed by unit
    int* gsym;                    // [n_units] symmetric GEMMs run for the unit
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
// two vector blocks (cap x VLD); they follow the S slots in the workspace.
__device__ __forceinline__ __half* c_ptr(const PEngine& e, __half* base, int slot, int buf, int& ldc) {
    if (buf < NBUF) { ldc = e.ld; return base + buf_off(e, slot, buf); }
    ldc = VLD;
    return base + (long long)e.S * e.slotsz + ((long long)slot * 2 + (buf - NBUF)) * ((long long)e.cap * VLD);
}

__device__ __forceinline__ float* pcols_ptr(const PEngine& e, int slot) { return e.pcols + (size_t)slot * e.cap * PCW; }

namespace pl {
__device__ __forceinline__ unsigned long long gtime() { return ptx::globaltimer_ns(); }
__device__ __forceinline__ void side_sync() { asm volatile("bar.sync 2, %0;" ::"n"(P_SIDE_THREADS) : "memory"); }
}  // namespace pl

// ------------------------------------------------------------------------------------------------
// Installing work on a slot (one thread; the slot has no other live work at that moment).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void p_install_side(const PEngine& e, int slot, int kind, int chunks) {
    __threadfence();
    *(volatile unsigned int*)&e.sclaim[slot] = ((unsigned)kind << 28) | ((unsigned)chunks << 14);
}
__device__ __forceinline__ void p_install_elem(const PEngine& e, int slot, int elem_kind) {
    __stcg(&e.slots[slot].elem_kind, elem_kind);
    p_install_side(e, slot, SK_ELEM, e.elem_chunks);
}

// Scaling alpha_k of sign iteration k (C-6b): X_{k+1} = 1/2 (alpha X_k)(3I - (alpha X_k)^2).
__device__ __forceinline__ float p_sign_alpha(const PEngine& e, const PSlot* s, int k) {
    return (k < e.n_sched && !__ldcg(&s->noboost)) ? e.alpha_sched[k] : 1.f;
}

__device__ __forceinline__ int p_tiles_of(const PEngine& e, int ntm, int flags) {
    if (flags & OPF_NARROW) return ntm;
    if ((flags & OPF_SYM) && e.sym_tiles) return ntm * (ntm + 1) / 2;
    return ntm * ntm;
}

__device__ __forceinline__ void p_install_gemm(const PEngine& e, int slot, int kind) {
    PSlot* s = &e.slots[slot];
    const int xcur = __ldcg(&s->xcur), ycur = __ldcg(&s->ycur), zcur = __ldcg(&s->zcur), xnext = __ldcg(&s->xsum) - xcur;
    const int k = __ldcg(&s->sign_iters);
    const bool first = k == 0;
    const int symx = e.lowdin ? OPF_SYM : 0;                                                       // the sign iterates are symmetric in the Loewdin form only
    int a = 0, b = 0, c = 0, flags = 0;
    float c_out = 1.f, alpha_res = 1.f, beta = 0.f;
    switch (kind) {
        case OP_INV_G1: a = 0; b = ycur; c = 4; c_out = -1.f; beta = 2.f; flags = OPF_RES | OPF_SYM; break;     // R = 2I - S Y
        case OP_INV_G2: a = ycur; b = 4; c = 5 - ycur; flags = OPF_SYM; break;                                   // Y <- Y R
        case OP_AMAT:                                                                                            // A = Y H0 - mu I (A0 = Y H0 with several trial mu)
            a = ycur; b = 1; 
            if (e.n_mu > 1) { c = 5; __stcg(&s->abuf, 5); } else { c = 0; beta = -e.mu[0]; }
            break;
        case OP_SIGN_G1: {                                                                          // T = 3I - alpha^2 X^2
            const float al = p_sign_alpha(e, s, k);
            alpha_res = first ? __ldcg(&s->alpha1) : 1.f;                                           // X0 = A / rho is never stored
            a = xcur; b = xcur; c = 4; c_out = -al * al * alpha_res; beta = 3.f; flags = OPF_RES | symx;
        } break;
        case OP_SIGN_G2: {                                                                          // X <- alpha/2 X T
            const float al = p_sign_alpha(e, s, k);
            a = xcur; b = 4; c = xnext; c_out = al * (first ? __ldcg(&s->alpha2) : 0.5f); flags = symx;
        } break;
        case OP_POW_S:
        case OP_POW_A: {                                                                            // V <- alpha M V
            const int st = __ldcg(&s->pow_step);
            a = __ldcg(&s->pow_buf); b = st == 0 ? NMAP - 1 : NBUF + ((st - 1) & 1); c = NBUF + (st & 1);
            c_out = alpha_res = __ldcg(&s->pow_alpha); flags = OPF_RES | OPF_NARROW;
        } break;
        case OP_DCOLS: a = xcur; b = e.lowdin ? zcur : ycur; c = 0; flags = OPF_NARROW; break;      // P = X Y[:, cols(i)]  (Loewdin: X Z[:, cols(i)])
        case OP_DCOLS2: a = zcur; b = NBUF; c = 0; flags = OPF_NARROW; break;                       // P = Z W, W = 1/2 (Z[:, cols] - X Z[:, cols])
        // ---- Loewdin form (C-21): Y0 = S / rho, Z0 = I ----
        case OP_LW_Y1: a = 0; b = 4; c = 2; c_out = 1.f / __ldcg(&s->rho_s); flags = OPF_SYM; break;              // Y1 = Y0 T0
        case OP_LW_G1: a = zcur; b = ycur; c = 4; c_out = -0.5f; beta = 1.5f; flags = OPF_RES | OPF_SYM; break;   // T = 1/2 (3I - Z Y)
        case OP_LW_G2: a = ycur; b = 4; c = 2 - ycur; flags = OPF_SYM; break;                                     // Y <- Y T
        case OP_LW_G3: a = 4; b = zcur; c = 8 - zcur; flags = OPF_SYM; break;                                     // Z <- T Z
        case OP_LW_HZ: a = 1; b = zcur; c = 0; break;                                                             // M = H0 Z
        case OP_LW_HT:                                                                                            // Ht = Z M / rho - mu I
            a = zcur; b = 0; c_out = 1.f / __ldcg(&s->rho_s); flags = OPF_SYM;
            if (e.n_mu > 1) { c = 8 - zcur; __stcg(&s->abuf, 8 - zcur); } else { c = 2; beta = -e.mu[0]; }
            break;
        default: break;
    }
    __stcg(reinterpret_cast<int4*>(&s->op_kind), make_int4(kind, a, b, c));
    __stcg(reinterpret_cast<float4*>(&s->c_out), make_float4(c_out, alpha_res, beta, __int_as_float(flags)));
    const unsigned long long tiles = (unsigned long long)p_tiles_of(e, __ldcg(&s->ntm), flags);
    const int seq = __ldcg(&s->op_seq) + 1;                        // generation of the claim word: a scheduler that cached the op's record
    __stcg(&s->op_seq, seq);                                       // sees when the word belongs to a newer op
    __threadfence();
    *(volatile unsigned long long*)&e.gclaim[slot] = ((unsigned long long)(seq & 0xFFFFFF) << 40) | (tiles << 20);
}

// Starts the block power iteration on buffer `buf` (S_sub or the X0 buffer): V0 = the shared +-1 start block.
__device__ __forceinline__ void p_start_power(const PEngine& e, int slot, int kind, int buf) {
    PSlot* s = &e.slots[slot];
    __stcg(&s->pow_step, 0);
    __stcg(&s->pow_norm2, (float)NVC * (float)__ldcg(&s->n));
    __stcg(&s->pow_alpha, 1.f);
    __stcg(&s->pow_g, 1.f);
    __stcg(&s->pow_buf, buf);
    p_install_gemm(e, slot, kind);
}

// L2 residency: a slot's iterates (X, T, Y: ~3-4 n^2 FP16) are re-read by every GEMM of its chain, so only
// as many slots as fit in L2 together may be inside the heavy phases (inverse iterations .. sign iterations)
// at once. A slot that is ready to enter takes a token or parks; a slot that leaves returns its token and wakes a
// parked slot if a token is free.
// A slot takes a token twice: for the inverse iterations .. A (resume == 0) and, after the power iteration for
// rho(A) - dependent 16-column tile passes that would hold the token idle - for the sign iterations (resume == 1).
__device__ __forceinline__ void p_enter_heavy_now(const PEngine& e, int slot) {
    PSlot* s = &e.slots[slot];
    if (__ldcg(&s->resume) == 0) {
        __stcg(&s->inv_iters, 1);
        if (e.lowdin) { __stcg(&s->ycur, 2); __stcg(&s->zcur, 3); p_install_gemm(e, slot, OP_LW_Y1); }
        else { __stcg(&s->ycur, 2); p_install_gemm(e, slot, OP_INV_G1); }
    } else {
        p_install_gemm(e, slot, OP_SIGN_G1);
    }
}
// Token count without transient overshoot (a failed atomicAdd-and-undo could make a concurrent waker give up).
__device__ __forceinline__ bool p_token_acquire(const PEngine& e) {
    int old = *(volatile int*)e.heavy;
    while (old < e.g_max) {
        const int prev = atomicCAS(e.heavy, old, old + 1);
        if (prev == old) return true;
        old = prev;
    }
    return false;
}
// Returns a token, then wakes a parked slot if a token can be taken again. Every release is followed by a scan, and a
// slot parks BEFORE its last attempt to take a token, so a parked slot is always seen by the release that frees the
// token it failed to get.
__device__ __forceinline__ void p_token_release(const PEngine& e) {
    atomicSub(e.heavy, 1);
    for (;;) {
        __threadfence();
        int found = -1;
        for (int s = 0; s < e.S; ++s)
            if (*(volatile int*)&e.parked[s] == 1) { found = s; break; }
        if (found < 0) return;
        if (!p_token_acquire(e)) return;              // every token is held: its holder wakes the parked slot when it leaves
        if (atomicCAS(&e.parked[found], 1, 0) == 1) { __threadfence(); p_enter_heavy_now(e, found); return; }
        atomicSub(e.heavy, 1);                        // somebody else admitted that slot: give the token back and look again
    }
}
__device__ __forceinline__ void p_enter_heavy(const PEngine& e, int slot) {
    if (p_token_acquire(e)) { p_enter_heavy_now(e, slot); return; }
    __threadfence();
    atomicExch(&e.parked[slot], 1);
    __threadfence();
    // a token may have been returned between the failed attempt and the parking: try once more
    if (p_token_acquire(e)) {
        if (atomicCAS(&e.parked[slot], 1, 0) == 1) { p_enter_heavy_now(e, slot); return; }
        p_token_release(e);                           // a leaving slot admitted this one meanwhile (with its own token)
    }
}
__device__ __forceinline__ void p_leave_heavy(const PEngine& e, int) { p_token_release(e); }

// Takes the next atom of the feed into the slot and installs its gather (phase NEW). Returns false when
// the feed is exhausted (the slot stays free).
__device__ __forceinline__ bool p_refill(const PEngine& e, int slot) {
    if (*(volatile int*)e.next_atom >= e.a_end) return false;
    const int fpos = atomicAdd(e.next_atom, 1);                         // a unit of the feed
    if (fpos >= e.a_end) return false;
    const int a = e.feed ? e.feed[fpos] : fpos;
    PSlot* s = &e.slots[slot];
    const int n = e.udim[a], n16 = (n + 15) & ~15;
    const int ntm = (n16 + BM - 1) / BM;
    const int nset = (int)(e.sv.uset_ptr[a + 1] - e.sv.uset_ptr[a]);
    int m0 = (int)e.sv.unit_ptr[a];
    const int m1 = (int)e.sv.unit_ptr[a + 1];
    while (m0 + 1 < m1 && (e.sv.unit_mem[m0] < e.atom_lo || e.sv.unit_mem[m0] >= e.atom_hi)) ++m0;   // the feed holds units with a member in range
    const int atom = e.sv.unit_mem[m0];
    __stcg(reinterpret_cast<int4*>(&s->atom), make_int4(atom, n, n16, e.upos[atom]));
    __stcg(reinterpret_cast<int4*>(&s->nbi), make_int4(e.at.nb[atom], ntm, nset, a));
    __stcg(reinterpret_cast<int4*>(&s->inv_iters), make_int4(0, 0, 0, 0));            // inv, sign, conv, xcur
    __stcg(reinterpret_cast<int4*>(&s->ycur), make_int4(2, 0, 0, 0));                 // ycur, status, gemm_count, tiles_done
    __stcg(reinterpret_cast<float4*>(&s->res_acc), make_float4(0.f, 1e30f, 0.f, 0.f)); // res_acc, res_prev, res_last, rho_s
    __stcg(reinterpret_cast<float4*>(&s->rho_a), make_float4(0.f, 1.f, 0.5f, 0.f));    // rho_a, alpha1, alpha2, side_done
    __stcg(reinterpret_cast<int4*>(&s->noboost), make_int4(0, m0, m1, 3));             // noboost, mptr, mend, zcur
    __stcg(reinterpret_cast<int4*>(&s->xsum), make_int4(e.lowdin ? 3 : 1, 0, 0, 0));   // xsum, pow_buf, mu_idx, sym_count
    __stcg(&s->elem_kind, 0); __stcg(&s->abuf, 0);                                     // op_seq keeps counting across the slot's atoms
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
    e.gsym[a] = __ldcg(&s->sym_count);
    const bool more = p_refill(e, slot);
    if (!more) *(volatile unsigned int*)&e.sclaim[slot] = 0u;
    __threadfence();
    atomicAdd(e.finished, 1);
}

// The sign chain of the slot's current trial mu starts: state of the iteration, then the power iteration for rho on the
// X0 buffer (buffer 0 in the Eq. 6 form, 2 in the Loewdin form).
__device__ __forceinline__ void p_begin_sign_chain(const PEngine& e, int slot) {
    PSlot* s = &e.slots[slot];
    const int x0 = e.lowdin ? 2 : 0;
    __stcg(reinterpret_cast<int4*>(&s->inv_iters), make_int4(__ldcg(&s->inv_iters), 0, 0, x0));   // sign_iters, conv, xcur
    __stcg(&s->noboost, 0);
    __stcg(&s->res_prev, 1e30f);
    p_start_power(e, slot, OP_POW_A, x0);
}

// ------------------------------------------------------------------------------------------------
// GEMM side: called by the finisher of a CTA pair once per finished tile (after the pair's stores and residual
// atomics). The last report of the op runs the slot's transition (C-7) and installs what comes next.
// ------------------------------------------------------------------------------------------------
// Convergence rule C-7 on the residual r of an inverse-type (inv) or sign iteration. Returns true when the iteration
// is over (converged, stagnated at the rounding floor, diverged or capped); sets the status bits.
__device__ __forceinline__ bool p_converged(const PEngine& e, PSlot* s, bool inv, float r, float rp) {
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
    return ok || stagnated || diverged || capped;
}

__device__ __forceinline__ void p_tile_finished(const PEngine& e, int slot, int nreports) {
    PSlot* s = &e.slots[slot];
    __threadfence();
    const int prev = atomicAdd(&s->tiles_done, 1);
    if (prev != nreports - 1) return;
    __threadfence();
    __stcg(&s->tiles_done, 0);
    const int kind = __ldcg(&s->op_kind);
    const int flags = __ldcg(&s->op_flags);
    if (kind == OP_POW_S || kind == OP_POW_A) {
        // ||alpha M V_k||_F^2 from the fused reduction; rho estimate = growth of the Frobenius norm
        const float r_new = atomicExch(&s->res_acc, 0.0f);
        const float alpha = __ldcg(&s->pow_alpha);
        float est = sqrtf(r_new / __ldcg(&s->pow_norm2)) / alpha;
        if (!(est > 1e-20f) || !(est < 1e20f)) est = 1.f;
        const int step = __ldcg(&s->pow_step) + 1;
        const int P = kind == OP_POW_S ? e.p_s : e.p_a;
        // rho(A): the estimate approaches rho from below, and the fixed safety factor covers a dense spectrum edge, where
        // the growth est_k / est_{k-1} falls from step to step (1.03 -> 1.02 at steps 5 -> 6). An eigenvalue outside the
        // bulk enters the start block with weight 1 / n only: the estimate sits at the bulk's edge and then starts to
        // climb, the growth RISES. A scaled sign step on such an underestimate would flip that eigenvalue's sign and
        // nothing would flag it, so the iteration goes on while the growth is still large or rising (up to p_cap steps).
        bool unsettled = false;
        if (kind == OP_POW_A && step >= P && step >= 3 && step < e.p_cap) {
            const float g = est * alpha, gp = __ldcg(&s->pow_g);        // alpha = 1 / est_{k-1} from the second step on
            unsettled = g > 1.05f || (g > gp + 0.003f && g > 1.004f);
            if (unsettled) atomicAdd(&e.ctr[PC_POW_EXTRA], 1ull);
        }
        if (step >= 2) __stcg(&s->pow_g, est * alpha);
        if (step < P || unsettled) {
            __stcg(&s->pow_step, step);
            __stcg(&s->pow_norm2, r_new);
            __stcg(&s->pow_alpha, 1.f / est);                         // keeps ||V_k||_F at its starting magnitude
            p_install_gemm(e, slot, kind);
        } else if (kind == OP_POW_S) {
            __stcg(&s->rho_s, e.safety_s * est);
            p_install_elem(e, slot, e.lowdin ? EL_LW1 : EL_SCHULZ1);
        } else {
            const float rho = e.safety_a * est;
            __stcg(&s->rho_a, rho);
            __stcg(&s->alpha1, 1.f / (rho * rho));
            __stcg(&s->alpha2, 0.5f / rho);
            __stcg(&s->resume, 1);
            p_enter_heavy(e, slot);
        }
        return;
    }
    if (kind == OP_DCOLS) {                 // a skinny product, not one of the counted square GEMMs
        if (__ldcg(&s->resume) != 2) { __stcg(&s->resume, 2); p_leave_heavy(e, slot); }          // first member served: the chain is over
        if (e.lowdin) p_install_side(e, slot, SK_WCOLS, 1);
        else p_install_side(e, slot, SK_DCOLS, e.dcols_chunks);
        return;
    }
    if (kind == OP_DCOLS2) { p_install_side(e, slot, SK_DCOLS, e.dcols_chunks); return; }
    if ((flags & OPF_SYM) && e.sym_tiles) __stcg(&s->sym_count, __ldcg(&s->sym_count) + 1);
    else __stcg(&s->gemm_count, __ldcg(&s->gemm_count) + 1);
    if (kind == OP_INV_G1 || kind == OP_SIGN_G1 || kind == OP_LW_G1) {
        const bool inv = kind != OP_SIGN_G1;
        const float sum = atomicExch(&s->res_acc, 0.0f);
        const float r = sqrtf(sum / (float)__ldcg(&s->n));
        const float rp = __ldcg(&s->res_prev);
        __stcg(&s->res_prev, r);
        __stcg(&s->res_last, r);
        const bool conv = p_converged(e, s, inv, r, rp);
        if (!inv && conv && p_sign_alpha(e, s, __ldcg(&s->sign_iters)) != 1.f) {
            // X_k passed the test, but T was formed with alpha_k != 1 and a scaled step would move the spectrum
            // away from +-1 again: switch the scaling off for this matrix and form T = 3I - X_k^2 once more
            __stcg(&s->noboost, 1);
            __stcg(&s->res_prev, rp);
            p_install_gemm(e, slot, OP_SIGN_G1);
            return;
        }
        __stcg(&s->conv, conv ? 1 : 0);
        if (kind == OP_INV_G1) p_install_gemm(e, slot, OP_INV_G2);
        else if (kind == OP_SIGN_G1) p_install_gemm(e, slot, OP_SIGN_G2);
        else p_install_gemm(e, slot, conv ? OP_LW_G3 : OP_LW_G2);      // the last step needs Z only
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
    } else if (kind == OP_LW_Y1) {
        p_install_gemm(e, slot, OP_LW_G1);
    } else if (kind == OP_LW_G2) {
        __stcg(&s->ycur, 2 - __ldcg(&s->ycur));
        p_install_gemm(e, slot, OP_LW_G3);
    } else if (kind == OP_LW_G3) {
        __stcg(&s->inv_iters, __ldcg(&s->inv_iters) + 1);
        __stcg(&s->zcur, 8 - __ldcg(&s->zcur));
        if (__ldcg(&s->conv)) {
            __stcg(&s->conv, 0);
            __stcg(&s->res_prev, 1e30f);
            if (__ldcg(&s->status) & ST_NOTSPD) { p_leave_heavy(e, slot); p_retire(e, slot); }
            else p_install_gemm(e, slot, OP_LW_HZ);
        } else {
            p_install_gemm(e, slot, OP_LW_G1);
        }
    } else if (kind == OP_LW_HZ) {
        p_install_gemm(e, slot, OP_LW_HT);
    } else if (kind == OP_AMAT || kind == OP_LW_HT) {
        p_leave_heavy(e, slot);                                  // the token is not held across the power iteration
        if (e.n_mu > 1) p_install_elem(e, slot, EL_SHIFT);      // X0 buffer = A0 - mu_0 I, then the sign chain
        else p_begin_sign_chain(e, slot);
    } else if (kind == OP_SIGN_G2) {
        __stcg(&s->sign_iters, __ldcg(&s->sign_iters) + 1);
        __stcg(&s->xcur, __ldcg(&s->xsum) - __ldcg(&s->xcur));
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
__device__ __forceinline__ void p_scheduler(const G2Smem& sm, const PEngine& e, int lane) {
    int q = 0; uint32_t ph = 0;
    unsigned long long idle_ns = 0, ntiles = 0, overshoot = 0;
    const unsigned long long t_begin = pl::gtime();
    bool short_tiles = false;
    // tiles claimed and not yet published (lane 0): tiles [pend_t, pend_end) of the op whose record is cached below
    int pend_t = 0, pend_end = 0, pend_slot = 0, pend_nt = 0, pend_gen = -1;
    bool sticky_ok = false;
    int4 g0 = make_int4(0, 0, 0, 0), g1 = g0, o0 = g0;
    float4 o1 = make_float4(0.f, 0.f, 0.f, 0.f);
    unsigned long long ring_ns = 0, credit_ns = 0;
    const int scan_off = e.scan_rotate && e.S <= 96 ? (int)(((blockIdx.x >> 1) * 13u) % (unsigned)e.S) : 0;   // (the one-shot scan covers 96 slots)
    for (;;) {
        const unsigned long long tr0 = pl::gtime();
        if (!ptx::mbar_wait_cluster_patient(sm.ti_empty(q), ph ^ 1, e.abort_flag)) break;
        const unsigned long long tr1 = pl::gtime();
        ring_ns += tr1 - tr0;
        // Claim lazily: only when the producer has issued every load of the tile before and needs the next
        // record (it runs G2_STAGES k-blocks ahead of the MMA, which hides the claim). A pair that claimed
        // further ahead would hoard tiles of a GEMM that idle pairs could run at the same time, and the
        // slot's chain of dependent GEMMs would take that much longer.
        {
            // short tiles (k-loop of a few microseconds): the claim - slot scan, atomic, slot record - takes as long as the tile,
            // so the scheduler may be three tiles ahead of the producer's claim points instead of one
            const int credits = short_tiles ? 3 : 1;
            uint32_t spins = 0; unsigned long long t0 = 0;
            bool stalled = false;
            while ((int)((uint32_t)ntiles - ptx::ld_shared_volatile_u32(sm.want())) >= credits) {
                __nanosleep(32);
                if ((++spins & 0xFFFFu) == 0 && ptx::stalled(t0, e.abort_flag)) { stalled = true; break; }
            }
            if (stalled) break;
        }
        credit_ns += pl::gtime() - tr1;
        TileInfo ti{};
        int got = __shfl_sync(0xffffffffu, pend_t < pend_end ? 1 : 0, 0), tflags = 0;
        unsigned long long t_idle0 = 0;
        if (!got && sticky_ok) {
            // the next tile of the GEMM this pair took its last tile from: one atomic, no scan, and the op's record is still
            // in registers when the generation of the claim word is the cached one
            unsigned long long w = 0;
            if (lane == 0) w = atomicAdd(&e.gclaim[pend_slot], 1ull);
            w = __shfl_sync(0xffffffffu, w, 0);
            const int t = (int)(w & 0xFFFFFu), nt = (int)((w >> 20) & 0xFFFFFu), gen = (int)(w >> 40);
            if (t < nt) {
                if (lane == 0) {
                    if (gen != pend_gen) {
                        __threadfence();
                        const PSlot* s = &e.slots[pend_slot];
                        g0 = __ldcg(reinterpret_cast<const int4*>(&s->atom));
                        g1 = __ldcg(reinterpret_cast<const int4*>(&s->nbi));
                        o0 = __ldcg(reinterpret_cast<const int4*>(&s->op_kind));
                        o1 = __ldcg(reinterpret_cast<const float4*>(&s->c_out));
                        pend_gen = gen;
                    }
                    pend_t = t; pend_end = t + 1; pend_nt = nt;
                }
                got = 1;
            } else {
                sticky_ok = false;
            }
        }
        while (!got) {
            // scan of the claim table in slot order: all words of a lane are loaded before the first ballot
            // (scan_off: with rotated scanning every pair starts at its own slot, so the claims of the 74 pairs spread over
            // the claim words instead of queueing on the first one)
            unsigned long long w3[3];
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                const int idx = 32 * r + lane;
                int sidx = idx + scan_off;
                if (sidx >= e.S) sidx -= e.S;
                w3[r] = idx < e.S ? *(volatile unsigned long long*)&e.gclaim[sidx] : 0ull;
            }
            int found = -1;
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                const bool avail = (unsigned)(w3[r] & 0xFFFFFu) < (unsigned)((w3[r] >> 20) & 0xFFFFFu);
                const unsigned m = __ballot_sync(0xffffffffu, avail);
                if (m && found < 0) {
                    found = 32 * r + __ffs(m) - 1 + scan_off;
                    if (found >= e.S) found -= e.S;
                }
            }
            for (int base = 96; base < e.S && found < 0; base += 32) {      // more than 96 slots (never by default)
                const int sidx = base + lane;
                const unsigned long long w = sidx < e.S ? *(volatile unsigned long long*)&e.gclaim[sidx] : 0ull;
                const bool avail = (unsigned)(w & 0xFFFFFu) < (unsigned)((w >> 20) & 0xFFFFFu);
                const unsigned m = __ballot_sync(0xffffffffu, avail);
                if (m) found = base + __ffs(m) - 1;
            }
            if (found >= 0) {
                // one tile per claim (three per claim for GEMMs of at most nine tiles was measured on cfg1: no faster without
                // combination, slower in the Loewdin form - the tiles of a GEMM should spread over pairs, not queue on one)
                unsigned long long w = 0;
                if (lane == 0) w = atomicAdd(&e.gclaim[found], 1ull);
                w = __shfl_sync(0xffffffffu, w, 0);
                const int t = (int)(w & 0xFFFFFu), nt = (int)((w >> 20) & 0xFFFFFu);
                if (t < nt) {
                    if (lane == 0) {
                        __threadfence();
                        const PSlot* s = &e.slots[found];
                        g0 = __ldcg(reinterpret_cast<const int4*>(&s->atom));     // atom n n16 pos
                        g1 = __ldcg(reinterpret_cast<const int4*>(&s->nbi));      // nbi ntm nset unit
                        o0 = __ldcg(reinterpret_cast<const int4*>(&s->op_kind));
                        o1 = __ldcg(reinterpret_cast<const float4*>(&s->c_out));
                        pend_t = t; pend_end = t + 1; pend_nt = nt; pend_gen = (int)(w >> 40);
                    }
                    pend_slot = found;
                    sticky_ok = e.scan_rotate != 0;
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
        if (got && lane == 0) {
            int t = pend_t++;
            const int flags = __float_as_int(o1.w), ntm = g1.y;
            ti.slot = pend_slot;
            tflags = TI_VALID;
            if (flags & OPF_NARROW) {
                ti.m0 = t * BM;
                tflags |= TI_PLAIN;
                if (o0.x == OP_DCOLS) { ti.n0 = g0.w & ~7; ti.bn = PCW; tflags |= TI_F32OUT; }   // D columns: the aligned window around pos(i)
                else if (o0.x == OP_DCOLS2) { ti.n0 = 0; ti.bn = PCW; tflags |= TI_F32OUT; }      // B operand: the W block
                else { ti.n0 = 0; ti.bn = NVC; }                                                  // power iteration
            } else {
                int tm, tn;
                if ((flags & OPF_SYM) && e.sym_tiles) {          // tiles on and above the diagonal, row by row
                    tm = 0;
                    while (t >= ntm - tm) { t -= ntm - tm; ++tm; }
                    tn = tm + t;
                    tflags |= tn > tm ? TI_MIRROR : TI_SYMDIAG;
                } else {
                    tm = t / ntm; tn = t - tm * ntm;
                }
                ti.m0 = tm * BM; ti.n0 = tn * BN; ti.bn = min(BN, g0.z - tn * BN);
                const int rleft = g0.z - tm * BM;                // rows of this row block
                if (e.trans_tiles && rleft < BM && tn < ntm - 1 && !(tflags & (TI_MIRROR | TI_SYMDIAG))) {
                    // ragged last row block, full-width column tile: computed transposed, the MMA's N = the rows left
                    tflags |= TI_TRANS; ti.bn = rleft;
                } else
                // the last row block when at most 128 rows are left: one M = 128 MMA per 16 k instead of M = 256
                if (rleft <= BM / 2 && (ti.bn & 31) == 0) tflags |= TI_HALF;
            }
            ti.n = g0.y; ti.n16 = g0.z; ti.nreports = pend_nt;
            ti.kind = o0.x; ti.a_buf = o0.y; ti.b_buf = o0.z; ti.c_buf = o0.w;
            ti.c_out = o1.x; ti.alpha_res = o1.y; ti.beta = o1.z; ti.want_res = flags & OPF_RES;
        }
        if (lane == 0) ti.valid = got ? tflags : 0;
        const uint32_t* w = reinterpret_cast<const uint32_t*>(&ti);
        uint32_t mine = 0;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const uint32_t v = __shfl_sync(0xffffffffu, w[i], 0);
            if (lane == i) mine = v;
        }
        short_tiles = __shfl_sync(0xffffffffu, ti.n16, 0) <= 768;
        if (lane < 16) {
#pragma unroll
            for (uint32_t rk = 0; rk < 2u; ++rk)
                ptx::st_async_u32(ptx::mapa(sm.tinfo(q), rk) + 4u * lane, mine, ptx::mapa(sm.ti_full(q), rk));
        }
        if (lane < 2) ptx::mbar_arrive_expect_tx_cluster(ptx::mapa(sm.ti_full(q), (uint32_t)lane), 64u);
        if (!got) break;
        if (++q == G2_NTI) { q = 0; ph ^= 1; }
    }
    if (lane == 0) {
        const unsigned long long t_end = pl::gtime();
        atomicAdd(&e.ctr[PC_TILES], ntiles);
        atomicAdd(&e.ctr[PC_SCHED_IDLE_NS], idle_ns);
        atomicAdd(&e.ctr[PC_SCHED_BUSY_NS], t_end - t_begin - idle_ns);
        atomicAdd(&e.ctr[PC_OVERSHOOT], overshoot);
        atomicAdd(&e.ctr[PC_SCHED_RING_NS], ring_ns);
        atomicAdd(&e.ctr[PC_SCHED_CREDIT_NS], credit_ns);
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
// Data path: the source blocks of a row-atom are contiguous runs of nb(j_a) x nb(j_b) values. Every warp loads G_NB blocks
// at a time with coalesced 8-byte loads, converts each value
// once (RN-even, C-13) into a shared-memory strip of the dense rows, and the strip leaves with 16-byte
// coalesced stores. Strips are G_STRIP_BYTES at most, so a row-atom of a very wide submatrix takes several passes over
// row sub-ranges of its blocks.
constexpr int G_STRIP_BYTES = 48 * 1024;
constexpr int G_NB = 2;                           // blocks a warp has in flight (8 loads per lane each)

template <typename TV>
__device__ void side_gather_chunk(const SysView& sv, const TV* __restrict__ S_vals, const TV* __restrict__ H_vals,
                                  __half* __restrict__ dstS, __half* __restrict__ dstH, int unit, int n, int n16, int ld,
                                  int chunk, int nchunks, unsigned char* sm, int tid, unsigned long long* bytes) {
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
                // ---- the strip leaves with 16-byte stores ----
                {
                    const uint4* s4 = reinterpret_cast<const uint4*>(strip);
                    for (int q = tid; q < nr * vpr; q += P_SIDE_THREADS) {
                        const int rr = q / vpr, v = q - rr * vpr;
                        *reinterpret_cast<uint4*>(dst + (long long)(row0 + r0 + rr) * ld + v * 8) = s4[q];
                    }
                }
                pl::side_sync();
            }
        }
    }
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

// Elementwise task, rows [r_lo, r_hi) of n16: dst = d I - sc src inside [0, n)^2, zero in the pad strip; dst2 (nullable)
// receives the same values. First Schulz step Y1 = (2/rho) I - S / rho^2 (C-8), first coupled Newton-Schulz
// step T0 = Z1 = 3/2 I - S / (2 rho) (C-21), diagonal shift A0 - mu I (C-20).
__device__ void side_elem_chunk(const __half* __restrict__ src, __half* __restrict__ dst, __half* __restrict__ dst2, int n, int n16, int ld,
                                float d, float sc, int chunk, int nchunks, int tid) {
    const int r_lo = (int)((long long)n16 * chunk / nchunks), r_hi = (int)((long long)n16 * (chunk + 1) / nchunks);
    const int ppr = n16 >> 3;
    const int total = (r_hi - r_lo) * ppr;
    constexpr int U = 4;
#pragma unroll 1
    for (int idx0 = tid; idx0 < total; idx0 += U * P_SIDE_THREADS) {
        uint4 u[U];
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int idx = idx0 + q * P_SIDE_THREADS;
            if (idx < total) {
                const int rl = idx / ppr, p = idx - rl * ppr;
                u[q] = __ldcg(reinterpret_cast<const uint4*>(src + (long long)(r_lo + rl) * ld + p * 8));
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
                st_half8(dst + (long long)r * ld + c0, f);
                if (dst2) st_half8(dst2 + (long long)r * ld + c0, f);
            }
        }
    }
}

// Loewdin form, between the two skinny products of a member's D columns: W[r, j] = 1/2 (Z[r, w0 + j] - P[r, j]) for the
// PCW columns of the aligned window w0 = pos & ~7, FP16 into the slot's first vector block (the B operand of OP_DCOLS2).
__device__ void side_wcols(const float* __restrict__ P, const __half* __restrict__ Z, __half* __restrict__ W, int n16, int ld, int w0, int tid) {
    for (int idx = tid; idx < n16 * (PCW / 8); idx += P_SIDE_THREADS) {
        const int r = idx / (PCW / 8), c0 = (idx - r * (PCW / 8)) * 8;
        const uint4 z = __ldcg(reinterpret_cast<const uint4*>(Z + (long long)r * ld + w0 + c0));
        const float4 p0 = __ldcg(reinterpret_cast<const float4*>(P + (size_t)r * PCW + c0));
        const float4 p1 = __ldcg(reinterpret_cast<const float4*>(P + (size_t)r * PCW + c0 + 4));
        const __half2* h = reinterpret_cast<const __half2*>(&z);
        const float2 z0 = __half22float2(h[0]), z1 = __half22float2(h[1]), z2 = __half22float2(h[2]), z3 = __half22float2(h[3]);
        float f[8] = {0.5f * (z0.x - p0.x), 0.5f * (z0.y - p0.y), 0.5f * (z1.x - p0.z), 0.5f * (z1.y - p0.w),
                      0.5f * (z2.x - p1.x), 0.5f * (z2.y - p1.y), 0.5f * (z3.x - p1.z), 0.5f * (z3.y - p1.w)};
        st_half8(W + (long long)r * VLD + c0, f);
    }
}

// a6 + a7, one chunk of the values of output row i (slot (i, j) holds (D_ji)^T, C-10):
// D_sub[r, pos + c] = ysc Y[r, pos + c] + psc P[r, c] with P from the skinny tensor tiles (Eq. 6 form: 1/2 (Y - X Y[:, cols]),
// Loewdin form: Z W / rho_s), and the energy partial sum <D_ji, H0_ji> in FP64 (Eq. 4). One thread per
// output value, in output order: the block-CSR arrays (D out, H0 in) are touched with coalesced accesses, the small
// L2-resident operands (Y columns, P) with scattered ones. D_vals == nullptr: only the partial sums (count_only).
template <typename TV, typename TD>
__device__ void side_dcols_chunk(const SysView& sv, const float* __restrict__ P, const __half* __restrict__ Y, float ysc, float psc,
                                 const TV* __restrict__ H_vals, const TV* __restrict__ S_vals, TD* __restrict__ D_vals, double* e_acc,
                                 double* q_acc, int atom, int n_own, int ld, int pos, int nbi, int chunk, int nchunks, unsigned char* sm, int tid) {
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
        float d = psc * __ldcg(P + (size_t)r * PCW + (pos & 7) + c);
        if (ysc != 0.f) d = fmaf(ysc, __half2float(__ldcg(Y + (long long)r * ld + pos + c)), d);
        if (D_vals) D_vals[o] = (TD)d;
        e_part += (double)d * (double)H_vals[o];
        q_part += (double)d * (double)S_vals[o];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { e_part += __shfl_xor_sync(0xffffffffu, e_part, o); q_part += __shfl_xor_sync(0xffffffffu, q_part, o); }
    if ((tid & 31) == 0 && e_part != 0.0) atomicAdd(e_acc, e_part);
    if ((tid & 31) == 0 && q_part != 0.0) atomicAdd(q_acc, q_part);
}

// ------------------------------------------------------------------------------------------------
// Side group main loop.
// ------------------------------------------------------------------------------------------------
__device__ void p_side_loop(const PEngine& e, unsigned char* sm, int tid) {
    __shared__ int s_ctl[4];                      // slot, kind, chunk, nchunks
    const int warp = tid >> 5, lane = tid & 31;
    unsigned long long busy_ns[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tasks[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (;;) {
        if (warp == 0) {
            int slot = -1, kind = -1, chunk = 0, nch = 0;
            for (;;) {
                int found = -1;
                for (int base = 0; base < e.S; base += 32) {
                    const int sidx = base + lane;
                    const unsigned w = sidx < e.S ? *(volatile unsigned int*)&e.sclaim[sidx] : 0u;
                    const bool avail = (w & 0x3FFFu) < ((w >> 14) & 0x3FFFu);
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
        const int4 g1 = __ldcg(reinterpret_cast<const int4*>(&s->nbi));      // nbi ntm nset unit
        const int atom = g0.x, n = g0.y, n16 = g0.z, pos = g0.w, nbi = g1.x;
        const int mu_idx = __ldcg(&s->mu_idx);
        switch (kind) {
            case SK_GATHER: {
                __half* dS = e.base + buf_off(e, slot, 0);
                __half* dH = e.base + buf_off(e, slot, 1);
                if (e.val_f64) side_gather_chunk<double>(e.sv, (const double*)e.S_vals, (const double*)e.H_vals, dS, dH, g1.w, n, n16, e.ld, chunk, nch, sm, tid, &e.ctr[PC_SIDE_BYTES + SK_GATHER]);
                else side_gather_chunk<float>(e.sv, (const float*)e.S_vals, (const float*)e.H_vals, dS, dH, g1.w, n, n16, e.ld, chunk, nch, sm, tid, &e.ctr[PC_SIDE_BYTES + SK_GATHER]);
            } break;
            case SK_ELEM: {
                const int ek = __ldcg(&s->elem_kind);
                const float rho = __ldcg(&s->rho_s);
                if (ek == EL_SCHULZ1)
                    side_elem_chunk(e.base + buf_off(e, slot, 0), e.base + buf_off(e, slot, 2), nullptr, n, n16, e.ld, 2.f / rho, 1.f / (rho * rho), chunk, nch, tid);
                else if (ek == EL_LW1)
                    side_elem_chunk(e.base + buf_off(e, slot, 0), e.base + buf_off(e, slot, 4), e.base + buf_off(e, slot, 3), n, n16, e.ld, 1.5f, 0.5f / rho, chunk, nch, tid);
                else
                    side_elem_chunk(e.base + buf_off(e, slot, __ldcg(&s->abuf)), e.base + buf_off(e, slot, e.lowdin ? 2 : 0), nullptr, n, n16, e.ld, -e.mu[mu_idx], -1.f, chunk, nch, tid);
            } break;
            case SK_WCOLS: {
                int ldw;
                __half* W = c_ptr(e, e.base, slot, NBUF, ldw);
                side_wcols(pcols_ptr(e, slot), e.base + buf_off(e, slot, __ldcg(&s->zcur)), W, n16, e.ld, pos & ~7, tid);
            } break;
            case SK_DCOLS: {
                const float* P = pcols_ptr(e, slot);
                const __half* Y = e.base + buf_off(e, slot, __ldcg(&s->ycur));
                const float ysc = e.lowdin ? 0.f : 0.5f, psc = e.lowdin ? 1.f / __ldcg(&s->rho_s) : -0.5f;
                double* e_acc = e.count_only ? &e.e_mu[mu_idx] : &e.e_atom[atom];
                double* q_acc = e.count_only ? &e.nelec_mu[mu_idx] : &e.q_atom[atom];
                void* Dv = e.count_only ? nullptr : e.D_vals;
                if (e.val_f64) {
                    if (e.d_f64) side_dcols_chunk<double, double>(e.sv, P, Y, ysc, psc, (const double*)e.H_vals, (const double*)e.S_vals, (double*)Dv, e_acc, q_acc, atom, e.adim[atom], e.ld, pos, nbi, chunk, nch, sm, tid);
                    else side_dcols_chunk<double, float>(e.sv, P, Y, ysc, psc, (const double*)e.H_vals, (const double*)e.S_vals, (float*)Dv, e_acc, q_acc, atom, e.adim[atom], e.ld, pos, nbi, chunk, nch, sm, tid);
                } else {
                    if (e.d_f64) side_dcols_chunk<float, double>(e.sv, P, Y, ysc, psc, (const float*)e.H_vals, (const float*)e.S_vals, (double*)Dv, e_acc, q_acc, atom, e.adim[atom], e.ld, pos, nbi, chunk, nch, sm, tid);
                    else side_dcols_chunk<float, float>(e.sv, P, Y, ysc, psc, (const float*)e.H_vals, (const float*)e.S_vals, (float*)Dv, e_acc, q_acc, atom, e.adim[atom], e.ld, pos, nbi, chunk, nch, sm, tid);
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
                    case SK_GATHER: p_start_power(e, slot, OP_POW_S, 0); break;
                    case SK_ELEM:
                        if (__ldcg(&s->elem_kind) == EL_SHIFT) p_begin_sign_chain(e, slot);
                        else p_enter_heavy(e, slot);
                        break;
                    case SK_WCOLS: p_install_gemm(e, slot, OP_DCOLS2); break;
                    case SK_DCOLS: {
                        const double nv = (double)(e.sv.blk_off[e.sv.row_ptr[atom + 1]] - e.sv.blk_off[e.sv.row_ptr[atom]]);
                        atomicAdd(&e.ctr[PC_SIDE_BYTES + SK_DCOLS],
                                  (unsigned long long)(nv * ((e.count_only ? 0 : (e.d_f64 ? 8 : 4)) + 2 * (e.val_f64 ? 8 : 4)) + (double)n * PCW * 4.0 + (double)n * nbi * 2.0));
                        // the next member of the unit takes its columns from the same X and Y; then the next trial mu
                        // restarts the sign chain on the resident A0; then the slot retires
                        int mp = __ldcg(&s->mptr) + 1;
                        const int mend = __ldcg(&s->mend);
                        while (mp < mend && (e.sv.unit_mem[mp] < e.atom_lo || e.sv.unit_mem[mp] >= e.atom_hi)) ++mp;
                        if (mp >= mend && mu_idx + 1 < e.n_mu) {
                            mp = (int)e.sv.unit_ptr[g1.w];
                            while (mp + 1 < mend && (e.sv.unit_mem[mp] < e.atom_lo || e.sv.unit_mem[mp] >= e.atom_hi)) ++mp;
                            const int nxt = e.sv.unit_mem[mp];
                            __stcg(&s->mptr, mp);
                            __stcg(&s->atom, nxt);
                            __stcg(&s->pos, e.upos[nxt]);
                            __stcg(&s->nbi, e.at.nb[nxt]);
                            __stcg(&s->mu_idx, mu_idx + 1);
                            p_install_elem(e, slot, EL_SHIFT);
                        } else if (mp < mend) {
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
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(P_THREADS, 1)
nolsm_persist_kernel(const __grid_constant__ PEngine e) {
    extern __shared__ uint8_t smem_raw[];
    G2Smem sm;
    sm.base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* side_sm = smem_raw + (sm.base - ptx::smem_u32(smem_raw)) + (G2_SMEM_BYTES - 1024);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();
    auto done = [&](const TileInfo& ti) { p_tile_finished(e, ti.slot, ti.nreports); };

    const uint32_t tmem_base = g2_setup(sm, warp, lane);

    if (warp < G2_EPI_WARPS) {
        g2_epilogue(sm, tmem_base, e, e.base, rank, warp, lane, e.maps, e.abort_flag, e.l2_store);
    } else if (warp == G2_WARP_SCHED) {
        if (rank == 0) p_scheduler(sm, e, lane);
    } else if (warp == G2_WARP_TMA) {
        g2_producer(sm, e.maps, rank, lane, e.want_lead, e.abort_flag, e.l2_load);
    } else if (warp == G2_WARP_MMA) {
        if (rank == 0) g2_mma(sm, tmem_base, lane, e.abort_flag, &e.ctr[PC_MMA_NS]);
        else g2_finisher(sm, lane, done, e.abort_flag);
    } else {
        p_side_loop(e, side_sm, (int)threadIdx.x - G2_CTRL_THREADS);
    }
    g2_teardown(tmem_base, warp);
}

// Stand-alone launches of the side tasks (diagnostics: nolsm_gather_submatrix, and the HBM-bandwidth measurement of the
// gather and scatter code without the GEMMs, nolsm_side_task_bandwidth). The same device functions as in the
// persistent kernel, one side group (128 threads) per CTA.
// grid = (chunks, units): unit atoms[blockIdx.y] is gathered into slot blockIdx.y % nslots.
template <typename TV>
__global__ void __launch_bounds__(P_SIDE_THREADS) k_side_gather(SysView sv, const TV* S_vals, const TV* H_vals, __half* base,
                                                                long long slotsz, long long bufsz, int ld, const int* units,
                                                                const int* dims, int nslots, unsigned long long* bytes) {
    extern __shared__ unsigned char sm_dyn[];
    const int unit = units[blockIdx.y], n = dims[unit], n16 = (n + 15) & ~15;
    __half* dS = base + (long long)(blockIdx.y % nslots) * slotsz;
    side_gather_chunk<TV>(sv, S_vals, H_vals, dS, dS + bufsz, unit, n, n16, ld, blockIdx.x, gridDim.x, sm_dyn, threadIdx.x, bytes);
}
// grid = (chunks, atoms): the scatter task for atom atoms[blockIdx.y] (its own submatrix; P and Y of slot blockIdx.y % nslots).
template <typename TV, typename TD>
__global__ void __launch_bounds__(P_SIDE_THREADS) k_side_dcols(SysView sv, const float* pcols, const __half* base, long long slotsz,
                                                               long long ybuf_off, int cap, int ld, const int* atoms, const int* dims,
                                                               const int* pos, const int* nb, int nslots, const TV* H_vals,
                                                               const TV* S_vals, TD* D_vals, double* e_atom, double* q_atom) {
    extern __shared__ unsigned char sm_dyn[];
    const int atom = atoms[blockIdx.y], sl = blockIdx.y % nslots;
    side_dcols_chunk<TV, TD>(sv, pcols + (size_t)sl * cap * PCW, base + (long long)sl * slotsz + ybuf_off, 0.5f, -0.5f, H_vals, S_vals,
                             D_vals, &e_atom[atom], &q_atom[atom], atom, dims[atom], ld, pos[atom], nb[atom], blockIdx.x, gridDim.x,
                             sm_dyn, threadIdx.x);
}

}  // namespace nolsm
