// Device-side data structures of the NOLSM engine.
//
// The workspace is a fixed set of SLOTS; each slot holds NBUF square FP16 (or FP32) buffers of
// capacity cap x ld and evaluates one atom submatrix T_i(H0), T_i(S) at a time.
// A slot walks through the phases
//     NEW   gather + rho(S) power iteration + closed-form first Schulz step
//     INV   Schulz iterations  R = 2I - S Y,  Y <- Y R            (ref [14])
//     AMAT  A = S^-1 H0 - mu I                                   (Eq. 5/8)
//     PA    rho(A) power iteration (spectral scaling of X0)
//     SIGN  Newton-Schulz  T = 3I - X^2,  X <- 1/2 X T           (Eq. 6)
//     FIN   D columns of atom i, scatter, energy partial         (Eq. 4)
// and is refilled with the next atom when it finishes (continuous batching). All slots advance
// together in ROUNDS; a round is a fixed sequence of kernel launches (captured once as a CUDA graph)
// whose kernels act on the slots that were in the matching phase when the round began. Phase
// transitions, convergence tests and the refill are decided on the device; the host only replays the
// graph until the device reports that every atom is done.
//
// Zero-pad invariant: every buffer that is used as a GEMM operand holds exact zeros in rows and
// columns [n, n16) (n16 = n rounded up to 16). The TMA tensor maps describe the full slot capacity,
// the GEMM k-loop stops at n16, and every writer (gather, first Schulz step, GEMM epilogues) writes
// the zero strips, so nothing outside [0, n16)^2 is ever multiplied into a stored element.
#pragma once
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace nolsm {

constexpr int NBUF = 6;          // Eq. 6 form: B0 = S then X(even), B1 = H0 then X(odd), B2/B3 = Y ping-pong, B4 = R / T, B5 = A0 (several trial mu);
                                 // Loewdin form: B0 = S, Y, then H0 Z; B1 = H0 then X; B2 = Y then X; B3/B5 = Z ping-pong (the free one keeps Ht0); B4 = T
constexpr int NMAP = NBUF + 3;   // tensor maps per slot: the buffers, two vector blocks (power iteration, W of the Loewdin D columns), the shared start block
constexpr int NVC = 16;          // vectors of the block power iteration (one 16-column GEMM tile)
constexpr int PCW = 32;          // columns of an OP_DCOLS tile: cols(i) = [pos, pos + nb(i)) inside [pos & ~7, (pos & ~7) + 32), TMA boxes start 16-byte aligned
constexpr int VLD = 64;          // leading dimension of a vector block (one 128-byte row)
constexpr int BM = 256;          // GEMM tile rows (one CTA pair, tcgen05 cta_group::2)
constexpr int BN = 256;          // GEMM tile columns; the last tile of a row is n16 - 256 (ntn - 1) wide
constexpr int BK = 64;           // GEMM k-block (one 128-byte swizzle atom of fp16)
constexpr int MAX_SLOTS = 1024;

constexpr int ST_NOTSPD = 1;     // Schulz inverse iteration diverged / did not converge
constexpr int ST_NOCONV = 2;     // sign iteration hit max_sign_iters

enum Phase { PH_FREE = 0, PH_NEW, PH_INV, PH_AMAT, PH_PA, PH_SIGN, PH_FIN };
enum OpKind { OP_NONE = 0, OP_INV_G1, OP_INV_G2, OP_AMAT, OP_SIGN_G1, OP_SIGN_G2, OP_POW_S, OP_POW_A,
              OP_DCOLS,     // persistent engine: P = X Y[:, cols(i)] as one 32-column tile per 256 rows, FP32 out
              OP_DCOLS2,    // Loewdin form: P = Z W
              OP_LW_Y1, OP_LW_G1, OP_LW_G2, OP_LW_G3, OP_LW_HZ, OP_LW_HT };   // coupled Newton-Schulz for S^-1/2 and Ht = Z H0 Z (persist.cuh)

struct __align__(16) Slot {
    // geometry of the atom in the slot (written at refill)
    int atom, n, n16, pos, nbi, ntm, ntn, pad0;
    // phase machine
    int phase;       // current phase (advanced by the kernels of the running round)
    int snap;        // phase when the running round began; kernels gate on this
    int inv_iters, sign_iters, conv, xcur, ycur, status, gemm_count, tiles_done;
    float res_acc, res_prev, res_last, rho_s, rho_a, alpha1, alpha2, unused;
};

// What a slot does in GEMM launch L (0 or 1) of the running round:
//   C = sgn * alpha * (A B) + beta * I,  optionally res += || alpha A B - I ||_F^2
struct __align__(16) SlotOp {
    int kind, a_buf, b_buf, c_buf;
    float alpha, sgn, beta;
    int want_res;
    int tile_start, ntiles, pad0, pad1;
};

struct AtomArrays {               // per-atom inputs and results (device)
    const int* dim;
    const int* pos;
    const int* nb;
    int *inv, *sign, *status, *gemms;
    float *res, *rho;
};

enum { PF_FLOP_USEFUL = 0, PF_FLOP_PADDED, PF_GATHER_SRC, PF_GATHER_DENSE, PF_DCOLS_BYTES, PF_SUBMATS, PF_LEN };

struct Engine {
    Slot* slots;
    SlotOp* ops;                  // [2][S]
    int* ntiles;                  // [2] tiles of GEMM launch 0 / 1 of the running round
    int S, cap, ld;               // slots, slot capacity (rows), leading dimension (elements)
    long long bufsz, slotsz;      // elements per buffer / per slot
    float tol_inv, tol_sign, mu;
    int max_inv, max_sign, p_s, p_a;
    int* next_atom;               // atom feed [*next_atom, a_end)
    int a_end;
    int* finished;                // atoms finished so far
    double* prof;                 // [PF_LEN] counters of the profiled rounds
    int profiling;                // this round is a profiled (eager, per-launch timed) round
    volatile int* h_done;         // host-mapped copy of *finished
    AtomArrays at;
};

__device__ __forceinline__ long long buf_off(const Engine& e, int slot, int buf) {
    return (long long)slot * e.slotsz + (long long)buf * e.bufsz;
}
// Output buffer of a GEMM op and its leading dimension (the round engine only has the square buffers).
__device__ __forceinline__ __half* c_ptr(const Engine& e, __half* base, int slot, int buf, int& ldc) {
    ldc = e.ld;
    return base + buf_off(e, slot, buf);
}

// FP32 output block of OP_DCOLS tiles (persistent engine only).
__device__ __forceinline__ float* pcols_ptr(const Engine&, int) { return nullptr; }

// Tile id -> slot by binary search over SlotOp::tile_start (a slot with ntiles == 0 shares its
// tile_start with the next slot and is never returned for a valid tile).
__device__ __forceinline__ int find_slot(const SlotOp* ops, int S, int tile) {
    int lo = 0, hi = S - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (ops[mid].tile_start <= tile) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// Called by exactly one thread per finished tile, after the tile's stores and residual atomics. The
// thread that finishes the last tile of the slot's GEMM advances the slot's iteration state
// (DESIGN.md "Readings" C-7).
__device__ __forceinline__ void tile_finished(const Engine& e, int slot, const SlotOp& op) {
    Slot& s = e.slots[slot];
    __threadfence();
    const int prev = atomicAdd(&s.tiles_done, 1);
    if (prev != op.ntiles - 1) return;
    __threadfence();
    s.tiles_done = 0;
    s.gemm_count += 1;
    if (op.kind == OP_INV_G1 || op.kind == OP_SIGN_G1) {
        const bool inv = op.kind == OP_INV_G1;
        const float sum = atomicExch(&s.res_acc, 0.0f);
        const float r = sqrtf(sum / (float)s.n);
        const float rp = s.res_prev;
        s.res_prev = r;
        s.res_last = r;
        const float tol = inv ? e.tol_inv : e.tol_sign;
        const int iters = inv ? s.inv_iters : s.sign_iters;
        const int cap = inv ? e.max_inv : e.max_sign;
        const bool ok = r < tol;
        const bool stagnated = (r > 0.5f * rp) && (r < 4.f * tol) && iters > 0;   // rounding floor reached
        const bool diverged = !(r == r) || (iters > 1 && r > rp && r > 0.9f);
        const bool capped = iters + 1 >= cap;
        if (diverged || (capped && !ok && !stagnated)) s.status |= inv ? ST_NOTSPD : ST_NOCONV;
        s.conv = (ok || stagnated || diverged || capped) ? 1 : 0;
    } else if (op.kind == OP_INV_G2) {
        s.inv_iters += 1;
        s.ycur = 5 - s.ycur;
        if (s.conv) { s.conv = 0; s.res_prev = 1e30f; s.phase = (s.status & ST_NOTSPD) ? PH_FIN : PH_AMAT; }
    } else if (op.kind == OP_AMAT) {
        s.phase = PH_PA;
    } else if (op.kind == OP_SIGN_G2) {
        s.sign_iters += 1;
        s.xcur = 1 - s.xcur;
        if (s.conv) { s.conv = 0; s.phase = PH_FIN; }
    }
}

}  // namespace nolsm
