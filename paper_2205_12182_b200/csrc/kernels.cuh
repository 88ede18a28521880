// SIMT kernels of the NOLSM engine: round bookkeeping (refill, phase snapshot, GEMM op tables), the
// block-CSR gather, power-iteration mat-vecs for the spectral scaling, the
// closed-form first Schulz step, a plain FFMA grouped GEMM (true-FP32 validation mode and FP16
// debugging reference) and the fused D-columns + scatter + energy kernel (Eq. 4).
// Every kernel acts only on the slots whose phase snapshot matches (nolsm_device.cuh).
#pragma once
#include "nolsm_device.cuh"

namespace nolsm {

template <typename T> struct Num;
template <> struct Num<float> {
    __device__ static float to_f(float v) { return v; }
    __device__ static float from_f(float v) { return v; }
    __device__ static float from_d(double v) { return (float)v; }
};
template <> struct Num<__half> {
    __device__ static float to_f(__half v) { return __half2float(v); }
    __device__ static __half from_f(float v) { return __float2half_rn(v); }
    __device__ static __half from_d(double v) { return __double2half(v); }   // single RN-even rounding
};

// Device view of the assembled system (borrowed / owned arrays of the context).
struct SysView {
    const long long* row_ptr;     // [n_atoms + 1]
    const int* col_idx;           // [nnzb]
    const long long* blk_off;     // [nnzb + 1]
    const int* atom_nb;           // [n_atoms]
    const long long* nset_ptr;    // [n_atoms + 1] index sets N(i) (== row_ptr when nothing is filtered)
    const int* nset_atom;         // atoms of N(i), ascending
    const int* nset_slot;         // slot of block (i, j) for j in N(i)
    const int* nset_off;          // first row/column of atom j inside submatrix i
    // Units of the persistent engine: one dense submatrix serves the columns of all member atoms of a unit
    // (Eq. 9 / Eq. 10; C-19). Without combination unit u is atom u and these arrays alias
    // the per-atom ones.
    const long long* unit_ptr;    // [n_units + 1] members of unit u: unit_mem[unit_ptr[u] .. unit_ptr[u + 1])
    const int* unit_mem;
    const long long* uset_ptr;    // [n_units + 1] index set of the unit (union of its members' N(i), ascending)
    const int* uset_atom;
    const int* uset_off;          // first row/column of that atom inside the unit's matrix
    const int* nset_uoff;         // for atom i, j in N(i): first row of atom j inside the matrix of i's unit
};

// Tiles of one n16 x n16 GEMM: ntm x ntn tiles of BM x BN; the last tile column is exactly as wide as
// what is left (a multiple of 16), so no columns are padded; rows are padded to BM.
__host__ __device__ __forceinline__ void choose_tiling(int n16, int& ntm, int& ntn) {
    ntm = (n16 + BM - 1) / BM;
    ntn = (n16 + BN - 1) / BN;
}

// ---------------------------------------------------------------------------------------------
// Round begin (one CTA, one thread per slot): apply the deferred transitions of the finished round,
// refill free slots with the next atoms, snapshot the phases, build the op tables and tile prefix
// sums of the two GEMM launches of this round, publish the number of finished atoms to the host.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(MAX_SLOTS) k_round_begin(Engine e) {
    __shared__ int s_t0[MAX_SLOTS], s_t1[MAX_SLOTS];
    __shared__ double s_fl[2];
    const int slot = threadIdx.x;
    int t0 = 0, t1 = 0;
    SlotOp o0{}, o1{};
    if (threadIdx.x < 2) s_fl[threadIdx.x] = 0.0;
    __syncthreads();
    if (slot < e.S) {
        Slot& s = e.slots[slot];
        if (s.snap == PH_NEW && s.phase == PH_NEW) s.phase = PH_INV;
        else if (s.snap == PH_PA && s.phase == PH_PA) s.phase = PH_SIGN;
        else if (s.snap == PH_FIN && s.phase == PH_FIN) {
            const int a = s.atom;
            e.at.inv[a] = s.inv_iters; e.at.sign[a] = s.sign_iters; e.at.status[a] = s.status;
            e.at.gemms[a] = s.gemm_count; e.at.res[a] = s.res_last; e.at.rho[a] = s.rho_a;
            atomicAdd(e.finished, 1);
            s.phase = PH_FREE;
            s.atom = -1;
        }
        if (s.phase == PH_FREE && *(volatile int*)e.next_atom < e.a_end) {
            const int a = atomicAdd(e.next_atom, 1);
            if (a < e.a_end) {
                s.atom = a; s.n = e.at.dim[a]; s.n16 = (s.n + 15) & ~15; s.pos = e.at.pos[a]; s.nbi = e.at.nb[a];
                choose_tiling(s.n16, s.ntm, s.ntn);
                s.inv_iters = 0; s.sign_iters = 0; s.conv = 0; s.xcur = 0; s.ycur = 2; s.status = 0;
                s.gemm_count = 0; s.tiles_done = 0;
                s.res_acc = 0.f; s.res_prev = 1e30f; s.res_last = 0.f; s.rho_s = 0.f; s.rho_a = 0.f;
                s.alpha1 = 1.f; s.alpha2 = 0.5f;
                s.phase = PH_NEW;
            }
        }
        s.snap = s.phase;
        const int tiles = s.ntm * s.ntn;
        const bool first = s.sign_iters == 0;
        switch (s.phase) {
            case PH_INV:
                o0.kind = OP_INV_G1; o0.a_buf = 0; o0.b_buf = s.ycur; o0.c_buf = 4; o0.alpha = 1.f; o0.sgn = -1.f; o0.beta = 2.f; o0.want_res = 1;
                o1.kind = OP_INV_G2; o1.a_buf = s.ycur; o1.b_buf = 4; o1.c_buf = 5 - s.ycur; o1.alpha = 1.f; o1.sgn = 1.f; o1.beta = 0.f;
                t0 = t1 = tiles;
                break;
            case PH_AMAT:
                o0.kind = OP_AMAT; o0.a_buf = s.ycur; o0.b_buf = 1; o0.c_buf = 0; o0.alpha = 1.f; o0.sgn = 1.f; o0.beta = -e.mu;
                t0 = tiles;
                break;
            case PH_SIGN:
                o0.kind = OP_SIGN_G1; o0.a_buf = s.xcur; o0.b_buf = s.xcur; o0.c_buf = 4; o0.alpha = first ? s.alpha1 : 1.f; o0.sgn = -1.f; o0.beta = 3.f; o0.want_res = 1;
                o1.kind = OP_SIGN_G2; o1.a_buf = s.xcur; o1.b_buf = 4; o1.c_buf = 1 - s.xcur; o1.alpha = first ? s.alpha2 : 0.5f; o1.sgn = 1.f; o1.beta = 0.f;
                t0 = t1 = tiles;
                break;
            default: break;
        }
        o0.ntiles = t0; o1.ntiles = t1;
        if (e.profiling && (t0 || t1)) {
            const double n = s.n, ng = (t0 ? 1 : 0) + (t1 ? 1 : 0);
            atomicAdd(&s_fl[0], 2.0 * n * n * n * ng);
            atomicAdd(&s_fl[1], 2.0 * (double)(s.ntm * BM) * (double)s.n16 * (double)s.n16 * ng);
        }
    }
    s_t0[threadIdx.x] = t0; s_t1[threadIdx.x] = t1;
    __syncthreads();
    // inclusive Hillis-Steele scan over MAX_SLOTS entries
    for (int d = 1; d < MAX_SLOTS; d <<= 1) {
        const int a0 = threadIdx.x >= d ? s_t0[threadIdx.x - d] : 0;
        const int a1 = threadIdx.x >= d ? s_t1[threadIdx.x - d] : 0;
        __syncthreads();
        s_t0[threadIdx.x] += a0; s_t1[threadIdx.x] += a1;
        __syncthreads();
    }
    if (slot < e.S) {
        o0.tile_start = s_t0[slot] - t0; o1.tile_start = s_t1[slot] - t1;
        e.ops[slot] = o0; e.ops[e.S + slot] = o1;
    }
    if (threadIdx.x == 0) {
        e.ntiles[0] = s_t0[MAX_SLOTS - 1]; e.ntiles[1] = s_t1[MAX_SLOTS - 1];
        if (e.profiling) { atomicAdd(&e.prof[PF_FLOP_USEFUL], s_fl[0]); atomicAdd(&e.prof[PF_FLOP_PADDED], s_fl[1]); }
        *e.h_done = *(volatile int*)e.finished;
        __threadfence_system();
    }
}

// ---------------------------------------------------------------------------------------------
// a1: gather (phase NEW). grid = (row-atom chunks, S, 2): z = 0 -> T_i(S) into buffer 0, z = 1 ->
// T_i(H0) into buffer 1. One CTA builds the dense rows of one row-atom j_a of N(i) at a time: the slots
// (j_a, j_b) are found by binary search in CSR row j_a, rows are written coalesced (zeros where the
// pair has no block and in the pad strips [n, n16)).
// ---------------------------------------------------------------------------------------------
template <typename TV, typename T>
__global__ void __launch_bounds__(256) k_gather(Engine e, SysView sv, const TV* S_vals, const TV* H_vals, T* base,
                                                int max_nset) {
    const Slot& s = e.slots[blockIdx.y];
    if (s.snap != PH_NEW) return;
    extern __shared__ unsigned char sm_raw[];
    long long* s_boff = reinterpret_cast<long long*>(sm_raw);           // [max_nset] blk_off of (j_a, j_b) or -1
    int* s_off = reinterpret_cast<int*>(s_boff + max_nset);             // [max_nset + 1]
    unsigned short* s_colmap = reinterpret_cast<unsigned short*>(s_off + max_nset + 1);   // [cap]
    const TV* vals = blockIdx.z == 0 ? S_vals : H_vals;
    T* dst = base + buf_off(e, blockIdx.y, blockIdx.z);
    const int n = s.n, n16 = s.n16, ld = e.ld;
    const long long p0 = sv.nset_ptr[s.atom];
    const int cnt = (int)(sv.nset_ptr[s.atom + 1] - p0);
    for (int b = threadIdx.x; b < cnt; b += blockDim.x) {
        const int o = sv.nset_off[p0 + b];
        s_off[b] = o;
        const int nbb = sv.atom_nb[sv.nset_atom[p0 + b]];
        for (int c = 0; c < nbb; ++c) s_colmap[o + c] = (unsigned short)b;
    }
    if (threadIdx.x == 0) s_off[cnt] = n;
    __syncthreads();
    int nread = 0;
    for (int a = blockIdx.x; a < cnt; a += gridDim.x) {
        const int j = sv.nset_atom[p0 + a];
        const long long r0 = sv.row_ptr[j], r1 = sv.row_ptr[j + 1];
        for (int b = threadIdx.x; b < cnt; b += blockDim.x) {
            const int k = sv.nset_atom[p0 + b];
            long long lo = r0, hi = r1;
            while (lo < hi) {
                const long long mid = (lo + hi) >> 1;
                if (sv.col_idx[mid] < k) lo = mid + 1; else hi = mid;
            }
            s_boff[b] = (lo < r1 && sv.col_idx[lo] == k) ? sv.blk_off[lo] : -1;
        }
        __syncthreads();
        const int nbj = sv.atom_nb[j];
        const int row0 = s_off[a];
        const int total = nbj * n16;
        for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
            const int rr = idx / n16;
            const int c = idx - rr * n16;
            T out = Num<T>::from_f(0.f);
            if (c < n) {
                const int b = s_colmap[c];
                const long long bo = s_boff[b];
                if (bo >= 0) {
                    const int nbb = s_off[b + 1] - s_off[b];
                    out = Num<T>::from_d((double)vals[bo + (long long)rr * nbb + (c - s_off[b])]);
                    ++nread;
                }
            }
            dst[(long long)(row0 + rr) * ld + c] = out;
        }
        __syncthreads();
    }
    // zero rows [n, n16)
    if (blockIdx.x == 0)
        for (int idx = threadIdx.x; idx < (n16 - n) * n16; idx += blockDim.x) {
            const int rr = idx / n16, c = idx - rr * n16;
            dst[(long long)(n + rr) * ld + c] = Num<T>::from_f(0.f);
        }
    if (e.profiling) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nread += __shfl_xor_sync(0xffffffffu, nread, o);
        if ((threadIdx.x & 31) == 0 && nread) atomicAdd(&e.prof[PF_GATHER_SRC], (double)nread);
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            atomicAdd(&e.prof[PF_GATHER_DENSE], (double)n16 * n16);
            if (blockIdx.z == 0) atomicAdd(&e.prof[PF_SUBMATS], 1.0);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// a3: spectral scaling by power iteration, x_{k+1} = M (x_k / ||x_k||), rho ~ ||x_{k+1}||, on buffer 0
// (S in phase NEW, A in phase PA). vec: [2][S][ld] floats, nrm2: [P + 1][S].
// ---------------------------------------------------------------------------------------------
__global__ void k_vec_init(Engine e, float* vec, float* nrm2, int P) {
    const Slot& s = e.slots[blockIdx.y];
    if (s.snap != PH_NEW && s.snap != PH_PA) return;
    float* xv = vec + (size_t)blockIdx.y * e.ld;
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < s.n; c += gridDim.x * blockDim.x) {
        unsigned h = (unsigned)c * 2654435761u + 0x9E3779B9u * (unsigned)(s.atom + 1);
        h ^= h >> 15; h *= 0x2C1B3C6Du; h ^= h >> 12;
        xv[c] = (h & 1u) ? 1.f : -1.f;
    }
    if (blockIdx.x == 0 && threadIdx.x <= P) nrm2[(size_t)threadIdx.x * e.S + blockIdx.y] = threadIdx.x == 0 ? (float)s.n : 0.f;
}

template <typename T>
__global__ void __launch_bounds__(256) k_matvec(Engine e, const T* base, float* vec, float* nrm2, int it) {
    const Slot& s = e.slots[blockIdx.y];
    if (!((s.snap == PH_NEW && it < e.p_s) || (s.snap == PH_PA && it < e.p_a))) return;
    const T* M = base + buf_off(e, blockIdx.y, 0);
    const float* x = vec + ((size_t)(it & 1) * e.S + blockIdx.y) * e.ld;
    float* y = vec + ((size_t)((it + 1) & 1) * e.S + blockIdx.y) * e.ld;
    const float sc = rsqrtf(nrm2[(size_t)it * e.S + blockIdx.y]);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float part = 0.f;
    for (int r = blockIdx.x * 8 + warp; r < s.n; r += gridDim.x * 8) {
        const T* row = M + (long long)r * e.ld;
        float acc = 0.f;
        if (sizeof(T) == 2) {
            // 8 halves (16 B) per lane; ld is a multiple of 16 and columns [n, n16) are zero
            for (int c = lane * 8; c < s.n16; c += 256) {
                const uint4 u = *reinterpret_cast<const uint4*>(reinterpret_cast<const __half*>(row) + c);
                const __half2* h = reinterpret_cast<const __half2*>(&u);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float2 f = __half22float2(h[q]);
                    const int cc = c + 2 * q;
                    acc += f.x * (cc < s.n ? x[cc] : 0.f) + f.y * (cc + 1 < s.n ? x[cc + 1] : 0.f);
                }
            }
        } else {
            for (int c = lane; c < s.n; c += 32) acc += Num<T>::to_f(row[c]) * x[c];
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        acc *= sc;
        if (lane == 0) { y[r] = acc; part += acc * acc; }
    }
    if (lane == 0 && part != 0.f) atomicAdd(&nrm2[(size_t)(it + 1) * e.S + blockIdx.y], part);
}

// Phase NEW: rho_s = 1.05 ||x_P||, then the first Schulz step in closed form
//   Y0 = I / rho, Y1 = Y0 (2I - S Y0) = (2/rho) I - S / rho^2   (into buffer 2, zero pad strips).
// Phase PA: rho_a and the first-iteration scalings alpha1 = 1 / rho^2, alpha2 = 1 / (2 rho).
template <typename T>
__global__ void k_power_finish(Engine e, T* base, const float* nrm2) {
    Slot& s = e.slots[blockIdx.y];
    if (s.snap == PH_PA) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            float rho = 1.05f * sqrtf(nrm2[(size_t)e.p_a * e.S + blockIdx.y]);
            if (!(rho > 1e-20f)) rho = 1.f;
            s.rho_a = rho; s.alpha1 = 1.f / (rho * rho); s.alpha2 = 0.5f / rho;
        }
        return;
    }
    if (s.snap != PH_NEW) return;
    float rho = 1.05f * sqrtf(nrm2[(size_t)e.p_s * e.S + blockIdx.y]);
    if (!(rho > 1e-20f)) rho = 1.f;
    const T* S = base + buf_off(e, blockIdx.y, 0);
    T* Y = base + buf_off(e, blockIdx.y, 2);
    const float d = 2.f / rho, sc = 1.f / (rho * rho);
    const int n = s.n, n16 = s.n16;
    const int total = n16 * n16;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const int r = idx / n16, c = idx - r * n16;
        const long long o = (long long)r * e.ld + c;
        float v = 0.f;
        if (r < n && c < n) v = (r == c ? d : 0.f) - sc * Num<T>::to_f(S[o]);
        Y[o] = Num<T>::from_f(v);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) { s.rho_s = rho; s.inv_iters = 1; s.ycur = 2; }
}

// ---------------------------------------------------------------------------------------------
// Plain FFMA grouped GEMM with the same op-table semantics as the tcgen05 kernel.
// grid = (max tiles of 64 x 64 per slot, S); 256 threads, 4 x 4 outputs each.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) k_gemm_simt(Engine e, T* base, int launch) {
    const int slot = blockIdx.y;
    SlotOp op = e.ops[launch * e.S + slot];
    if (op.kind == OP_NONE) return;
    const Slot& s = e.slots[slot];
    const int n = s.n, n16 = s.n16, ld = e.ld;
    const int nt = (n16 + 63) / 64;
    if ((int)blockIdx.x >= nt * nt) return;
    op.ntiles = nt * nt;
    const int tm = blockIdx.x / nt, tn = blockIdx.x - tm * nt;
    const T* A = base + buf_off(e, slot, op.a_buf);
    const T* B = base + buf_off(e, slot, op.b_buf);
    T* C = base + buf_off(e, slot, op.c_buf);
    __shared__ float sA[16][64 + 4];
    __shared__ float sB[16][64 + 4];
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    float acc[4][4] = {};
    for (int k0 = 0; k0 < n; k0 += 16) {
        for (int q = threadIdx.x; q < 64 * 16; q += 256) {
            const int r = q >> 4, k = q & 15;                  // A tile: 64 rows x 16 k
            const int gr = tm * 64 + r, gk = k0 + k;
            sA[k][r] = (gr < n && gk < n) ? Num<T>::to_f(A[(long long)gr * ld + gk]) : 0.f;
            const int kb = q >> 6, c = q & 63;                 // B tile: 16 k x 64 cols
            const int gkb = k0 + kb, gc = tn * 64 + c;
            sB[kb][c] = (gkb < n && gc < n) ? Num<T>::to_f(B[(long long)gkb * ld + gc]) : 0.f;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            float a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) { a[i] = sA[k][ty * 4 + i]; b[i] = sB[k][tx * 4 + i]; }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }
    float rsum = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int r = tm * 64 + ty * 4 + i;
        if (r >= n16) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int c = tn * 64 + tx * 4 + j;
            if (c >= n16) continue;
            const float x = op.alpha * acc[i][j];
            const float delta = (r == c && r < n) ? 1.f : 0.f;
            if (op.want_res) { const float d = x - delta; rsum += d * d; }
            C[(long long)r * ld + c] = Num<T>::from_f(op.sgn * x + op.beta * delta);
        }
    }
    __shared__ float s_red[8];
    if (op.want_res) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) rsum += __shfl_xor_sync(0xffffffffu, rsum, o);
        if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = rsum;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (op.want_res) {
            float t = 0.f;
            for (int w = 0; w < 8; ++w) t += s_red[w];
            if (t != 0.f) atomicAdd(&e.slots[slot].res_acc, t);
        }
        tile_finished(e, slot, op);
    }
}

// ---------------------------------------------------------------------------------------------
// a6 + a7 (phase FIN): D_sub[:, cols(i)] = 1/2 (Y[:, cols] - X Y[:, cols])  (Eq. 8 with sign(A) = X,
// S^-1 = Y), scattered into slot (i, j) of the output as (D_ji)^T, and
// e_i = sum_j <D_ji, H0_ji> accumulated in FP64 (Eq. 4, H0 symmetric).
// grid = (row chunks, S); dynamic smem: int off[max_nset + 1], float Yc[n][nbi].
// ---------------------------------------------------------------------------------------------
template <typename T, typename TV, typename TD>
__global__ void __launch_bounds__(256) k_dcols_scatter(Engine e, SysView sv, const T* base, const TV* H_vals, const TV* S_vals, TD* D_vals,
                                                       double* e_atom, double* q_atom, int max_nset) {
    const int slot = blockIdx.y;
    const Slot& s = e.slots[slot];
    if (s.snap != PH_FIN || (s.status & ST_NOTSPD)) return;
    extern __shared__ unsigned char sm_raw[];
    int* s_off = reinterpret_cast<int*>(sm_raw);                         // [max_nset + 1]
    float* s_y = reinterpret_cast<float*>(s_off + max_nset + 1);        // [n][nbi]
    const T* X = base + buf_off(e, slot, s.xcur);
    const T* Y = base + buf_off(e, slot, s.ycur);
    const int n = s.n, nbi = s.nbi, ld = e.ld;
    const long long p0 = sv.nset_ptr[s.atom];
    const int cnt = (int)(sv.nset_ptr[s.atom + 1] - p0);
    for (int b = threadIdx.x; b < cnt; b += blockDim.x) s_off[b] = sv.nset_off[p0 + b];
    if (threadIdx.x == 0) s_off[cnt] = n;
    for (int idx = threadIdx.x; idx < n * nbi; idx += blockDim.x) {
        const int k = idx / nbi, c = idx - k * nbi;
        s_y[idx] = Num<T>::to_f(Y[(long long)k * ld + s.pos + c]);
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double e_part = 0.0, q_part = 0.0;
    for (int r = blockIdx.x * 8 + warp; r < n; r += gridDim.x * 8) {
        int lo = 0, hi = cnt - 1;                                   // atom of N(i) that owns row r
        while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (s_off[mid] <= r) lo = mid; else hi = mid - 1; }
        const int a = lo, bb = r - s_off[a], nbj = s_off[a + 1] - s_off[a];
        const long long out0 = sv.blk_off[sv.nset_slot[p0 + a]];
        const T* xrow = X + (long long)r * ld;
        for (int c0 = 0; c0 < nbi; c0 += 16) {
            const int nc = min(16, nbi - c0);
            float acc[16];
#pragma unroll
            for (int c = 0; c < 16; ++c) acc[c] = 0.f;
            for (int k = lane; k < n; k += 32) {
                const float x = Num<T>::to_f(xrow[k]);
                const float* yr = s_y + k * nbi + c0;
#pragma unroll
                for (int c = 0; c < 16; ++c) if (c < nc) acc[c] = fmaf(x, yr[c], acc[c]);
            }
#pragma unroll
            for (int c = 0; c < 16; ++c)
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
            float mine = 0.f;
#pragma unroll
            for (int c = 0; c < 16; ++c) if (lane == c) mine = acc[c];
            if (lane < nc) {
                const int c = c0 + lane;
                const float d = 0.5f * (s_y[r * nbi + c] - mine);
                const long long o = out0 + (long long)c * nbj + bb;      // slot (i, j_a): [c][bb] = D_sub[r, pos + c]
                D_vals[o] = (TD)d;
                e_part += (double)d * (double)H_vals[o];
                q_part += (double)d * (double)S_vals[o];
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { e_part += __shfl_xor_sync(0xffffffffu, e_part, o); q_part += __shfl_xor_sync(0xffffffffu, q_part, o); }
    if (lane == 0 && e_part != 0.0) atomicAdd(&e_atom[s.atom], e_part);
    if (lane == 0 && q_part != 0.0) atomicAdd(&q_atom[s.atom], q_part);
    if (e.profiling && blockIdx.x == 0 && threadIdx.x == 0) {
        const double nv = (double)(sv.blk_off[sv.row_ptr[s.atom + 1]] - sv.blk_off[sv.row_ptr[s.atom]]);
        atomicAdd(&e.prof[PF_DCOLS_BYTES], nv * (sizeof(TD) + sizeof(TV)) + ((double)n * n + (double)n * nbi) * sizeof(T));
    }
}

// C-1 filter: keep[s] = max(|H0 block|_max, |S block|_max) > eps (diagonal handled on the host)
template <typename TV>
__global__ void k_block_keep(const long long* blk_off, const TV* H_vals, const TV* S_vals, long long nnzb, double eps,
                             unsigned char* keep) {
    const long long s = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (s >= nnzb) return;
    const int lane = threadIdx.x & 31;
    double mx = 0.0;
    for (long long q = blk_off[s] + lane; q < blk_off[s + 1]; q += 32)
        mx = fmax(mx, fmax(fabs((double)H_vals[q]), fabs((double)S_vals[q])));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (lane == 0) keep[s] = mx > eps ? 1 : 0;
}

}  // namespace nolsm
