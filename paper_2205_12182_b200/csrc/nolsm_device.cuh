// Device-side data structures shared by the NOLSM kernels (gather, grouped GEMM chain, D columns).
//
// One "batch" is a set of atom submatrices T_i(H0), T_i(S) that live in the
// workspace at the same time; every matrix of the batch owns one fixed-size workspace slot holding
// NBUF square buffers. All matrix iterations (Schulz inverse, ref [14] PAPER.md:L217; Newton-Schulz
// sign, Eq. 6) are sequences of grouped GEMM launches over the batch; convergence is
// decided on the device by the epilogue of the GEMM that forms the residual.
#pragma once
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace nolsm {

constexpr int NBUF = 5;          // workspace buffers per matrix slot
constexpr int BM = 128;          // GEMM tile rows
constexpr int BK = 64;           // GEMM k-block (one 128-byte swizzle atom of fp16)

// status bits per submatrix (nolsm.h: NOLSM_MAT_*)
constexpr int ST_NOTSPD = 1;     // Schulz inverse iteration did not converge / diverged
constexpr int ST_NOCONV = 2;     // sign iteration hit max_sign_iters

// Per-matrix geometry of the current batch (device array, written at assemble time).
struct MatInfo {
    int n;            // true dimension n_i
    int ld;           // leading dimension (elements), multiple of 8
    int pos;          // first column of atom i inside its own submatrix
    int nbi;          // basis functions of atom i
    int tile_start;   // first tile id of this matrix in the batch tile list
    int ntn;          // tiles along N
    int bn;           // tile width along N (multiple of 16, <= 256)
    int atom;         // global atom id
    long long off;    // element offset of buffer 0 of this matrix in the workspace
    long long bufsz;  // elements per buffer (>= n * ld, multiple of 64)
};

// Mutable per-matrix iteration state (device, SoA, indexed by slot in the batch).
struct BatchState {
    float* res_acc;      // running sum of squares accumulated by the residual epilogue
    float* res_prev;     // residual of the previous iteration (||.||_F / sqrt(n))
    float* res_last;     // last residual measured
    float* rho_s;        // spectral-radius estimate of S_sub
    float* rho_a;        // spectral-radius estimate of A_sub
    float* alpha1;       // first sign iteration: 1 / rho_a^2
    float* alpha2;       // first sign iteration: 0.5 / rho_a
    int* tiles_done;     // tiles finished in the running launch
    int* inv_conv;       // residual passed in G1 of this iteration
    int* inv_done;       // inverse finished
    int* inv_iters;
    int* ybuf;           // buffer id holding S^-1 once inv_done
    int* sign_conv;
    int* sign_done;
    int* sign_iters;
    int* xbuf;           // buffer id holding sign(A) once sign_done
    int* status;         // ST_* bits
    int* gemm_count;     // executed square GEMMs (FLOP accounting)
};

enum FinishKind { FIN_NONE = 0, FIN_INV_G1, FIN_INV_G2, FIN_SIGN_G1, FIN_SIGN_G2, FIN_COUNT_ONLY };
enum GateKind { GATE_NONE = 0, GATE_INV_ACTIVE, GATE_SIGN_ACTIVE, GATE_INV_OK };

// One grouped GEMM launch: for every gated matrix m of the batch
//   C_m = sgn * alpha_m * (A_m B_m) + beta * I,   optionally res_m += || alpha_m A_m B_m - I ||_F^2
struct GemmOp {
    int nmat;
    int ntiles;
    const MatInfo* mats;
    BatchState st;
    int a_buf, b_buf, c_buf;     // buffer ids; a_buf == -1 -> per-matrix st.ybuf[m]
    float alpha;                 // scalar alpha, used when alpha_arr == nullptr
    const float* alpha_arr;
    float sgn;                   // +1 or -1
    float beta;
    int want_res;
    int gate;                    // GateKind
    int finish;                  // FinishKind
    float tol;
    int max_iters;
};

__device__ __forceinline__ bool gate_open(const GemmOp& op, int m) {
    switch (op.gate) {
        case GATE_INV_ACTIVE:  return op.st.inv_done[m] == 0;
        case GATE_SIGN_ACTIVE: return op.st.sign_done[m] == 0 && (op.st.status[m] & ST_NOTSPD) == 0;
        case GATE_INV_OK:      return (op.st.status[m] & ST_NOTSPD) == 0;
        default:               return true;
    }
}

// Tile id -> matrix index by binary search over MatInfo::tile_start.
__device__ __forceinline__ int find_matrix(const MatInfo* mats, int nmat, int tile) {
    int lo = 0, hi = nmat - 1;
    while (lo < hi) {
        int mid = (lo + hi + 1) >> 1;
        if (mats[mid].tile_start <= tile) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// Called by exactly one thread once per finished tile, after the tile's stores and residual
// atomics were issued and fenced. The thread that finishes the last tile of matrix m advances the
// matrix's iteration state (convergence test of SURVEY C-7 / DESIGN.md "Convergence").
__device__ __forceinline__ void tile_finished(const GemmOp& op, int m, int ntiles_m) {
    if (op.finish == FIN_NONE) return;
    __threadfence();
    int prev = atomicAdd(&op.st.tiles_done[m], 1);
    if (prev != ntiles_m - 1) return;
    __threadfence();
    op.st.tiles_done[m] = 0;
    atomicAdd(&op.st.gemm_count[m], 1);
    const BatchState& s = op.st;
    const float n = (float)op.mats[m].n;
    if (op.finish == FIN_INV_G1 || op.finish == FIN_SIGN_G1) {
        float sum = atomicExch(&s.res_acc[m], 0.0f);
        float r = sqrtf(sum / n);
        float rp = s.res_prev[m];
        s.res_prev[m] = r;
        s.res_last[m] = r;
        int* conv = (op.finish == FIN_INV_G1) ? s.inv_conv : s.sign_conv;
        int iters = (op.finish == FIN_INV_G1) ? s.inv_iters[m] : s.sign_iters[m];
        bool ok = r < op.tol;
        bool stagnated = (r > 0.5f * rp) && (r < 4.f * op.tol) && iters > 0;   // rounding floor reached
        bool diverged = !(r == r) || (iters > 1 && r > rp && r > 0.9f);
        bool capped = iters + 1 >= op.max_iters;
        if (diverged || (capped && !ok && !stagnated))
            atomicOr(&s.status[m], op.finish == FIN_INV_G1 ? ST_NOTSPD : ST_NOCONV);
        conv[m] = (ok || stagnated || diverged || capped) ? 1 : 0;
    } else if (op.finish == FIN_INV_G2) {
        s.inv_iters[m] += 1;
        if (s.inv_conv[m]) { s.inv_done[m] = 1; s.ybuf[m] = op.c_buf; }
    } else if (op.finish == FIN_SIGN_G2) {
        s.sign_iters[m] += 1;
        if (s.sign_conv[m]) { s.sign_done[m] = 1; s.xbuf[m] = op.c_buf; }
    }
}

}  // namespace nolsm
