// SIMT kernels of the NOLSM hot path: block-CSR gather, power-iteration
// mat-vecs for the spectral scaling, the elementwise first Schulz
// step, a plain FFMA grouped GEMM (true FP32 validation mode and FP16 debugging reference), and the
// fused D-columns + scatter + energy kernel (Eq. 4).
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
};

// ---------------------------------------------------------------------------------------------
// a1: gather.  grid = (row-atom chunks, nmat, 2): z = 0 -> T_i(S) into buffer 0, z = 1 -> T_i(H0)
// into buffer 1. One CTA builds the dense rows of one row-atom j_a of N(i) at a time: the slots
// (j_a, j_b) are found by binary search in CSR row j_a, rows are written coalesced (zeros where the
// pair has no block, and in the pad columns [n, ld)).
// ---------------------------------------------------------------------------------------------
template <typename TV, typename T>
__global__ void __launch_bounds__(256) k_gather(SysView sv, const MatInfo* mats, const TV* S_vals, const TV* H_vals,
                                                T* base, int max_nset, int max_ld, unsigned long long* src_elems) {
    extern __shared__ unsigned char sm_raw[];
    long long* s_boff = reinterpret_cast<long long*>(sm_raw);           // [max_nset] blk_off of (j_a, j_b) or -1
    int* s_off = reinterpret_cast<int*>(s_boff + max_nset);             // [max_nset + 1]
    unsigned short* s_colmap = reinterpret_cast<unsigned short*>(s_off + max_nset + 1);   // [max_ld]
    const MatInfo mi = mats[blockIdx.y];
    const TV* vals = blockIdx.z == 0 ? S_vals : H_vals;
    T* dst = base + mi.off + (long long)blockIdx.z * mi.bufsz;
    const long long p0 = sv.nset_ptr[mi.atom];
    const int cnt = (int)(sv.nset_ptr[mi.atom + 1] - p0);
    for (int b = threadIdx.x; b < cnt; b += blockDim.x) {
        const int o = sv.nset_off[p0 + b];
        s_off[b] = o;
        const int nbb = sv.atom_nb[sv.nset_atom[p0 + b]];
        for (int c = 0; c < nbb; ++c) s_colmap[o + c] = (unsigned short)b;
    }
    if (threadIdx.x == 0) s_off[cnt] = mi.n;
    __syncthreads();
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
        const int total = nbj * mi.ld;
        int nread = 0;
        for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
            const int rr = idx / mi.ld;
            const int c = idx - rr * mi.ld;
            T out = Num<T>::from_f(0.f);
            if (c < mi.n) {
                const int b = s_colmap[c];
                const long long bo = s_boff[b];
                if (bo >= 0) {
                    const int nbb = s_off[b + 1] - s_off[b];
                    out = Num<T>::from_d((double)vals[bo + (long long)rr * nbb + (c - s_off[b])]);
                    ++nread;
                }
            }
            dst[(long long)(row0 + rr) * mi.ld + c] = out;
        }
        if (src_elems) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) nread += __shfl_xor_sync(0xffffffffu, nread, o);
            if ((threadIdx.x & 31) == 0 && nread) atomicAdd(src_elems, (unsigned long long)nread);
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// per-batch state reset
// ---------------------------------------------------------------------------------------------
__global__ void k_state_init(BatchState st, int nmat) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= nmat) return;
    st.res_acc[m] = 0.f; st.res_prev[m] = 1e30f; st.res_last[m] = 0.f;
    st.rho_s[m] = 0.f; st.rho_a[m] = 0.f; st.alpha1[m] = 1.f; st.alpha2[m] = 0.5f;
    st.tiles_done[m] = 0; st.inv_conv[m] = 0; st.inv_done[m] = 0; st.inv_iters[m] = 0; st.ybuf[m] = 2;
    st.sign_conv[m] = 0; st.sign_done[m] = 0; st.sign_iters[m] = 0; st.xbuf[m] = 0; st.status[m] = 0;
    st.gemm_count[m] = 0;
}

// ---------------------------------------------------------------------------------------------
// a3: spectral scaling by power iteration.  x_{k+1} = M (x_k / ||x_k||), rho ~ ||x_{k+1}||.
// ---------------------------------------------------------------------------------------------
__global__ void k_vec_init(const MatInfo* mats, float* x, float* nrm2, int ldx) {
    const MatInfo mi = mats[blockIdx.y];
    float* xv = x + (size_t)blockIdx.y * ldx;
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < mi.n; c += gridDim.x * blockDim.x) {
        unsigned h = (unsigned)c * 2654435761u + 0x9E3779B9u * (unsigned)(mi.atom + 1);
        h ^= h >> 15; h *= 0x2C1B3C6Du; h ^= h >> 12;
        xv[c] = (h & 1u) ? 1.f : -1.f;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) nrm2[blockIdx.y] = (float)mi.n;
}

template <typename T>
__global__ void __launch_bounds__(256) k_matvec(const MatInfo* mats, const T* base, int buf, const float* xin,
                                                const float* nrm2_in, float* yout, float* nrm2_out, int ldx) {
    const MatInfo mi = mats[blockIdx.y];
    const T* M = base + mi.off + (long long)buf * mi.bufsz;
    const float* x = xin + (size_t)blockIdx.y * ldx;
    float* y = yout + (size_t)blockIdx.y * ldx;
    const float s = rsqrtf(nrm2_in[blockIdx.y]);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float part = 0.f;
    for (int r = blockIdx.x * 8 + warp; r < mi.n; r += gridDim.x * 8) {
        const T* row = M + (long long)r * mi.ld;
        float acc = 0.f;
        for (int c = lane; c < mi.n; c += 32) acc += Num<T>::to_f(row[c]) * x[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        acc *= s;
        if (lane == 0) { y[r] = acc; part += acc * acc; }
    }
    if (lane == 0 && part != 0.f) atomicAdd(&nrm2_out[blockIdx.y], part);
}

// which = 0: rho_s; which = 1: rho_a and the first-iteration scalings alpha1 = 1/rho^2, alpha2 = 1/(2 rho)
__global__ void k_rho_finish(BatchState st, const float* nrm2, int nmat, int which, float safety) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= nmat) return;
    float rho = sqrtf(nrm2[m]) * safety;
    if (!(rho > 1e-20f)) rho = 1.f;
    if (which == 0) st.rho_s[m] = rho;
    else { st.rho_a[m] = rho; st.alpha1[m] = 1.f / (rho * rho); st.alpha2[m] = 0.5f / rho; }
}

// ---------------------------------------------------------------------------------------------
// a2, first Schulz step in closed form: Y0 = I / rho, Y1 = Y0 (2I - S Y0) = (2/rho) I - S / rho^2.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void k_schulz_first(const MatInfo* mats, BatchState st, T* base, int s_buf, int y_buf) {
    const MatInfo mi = mats[blockIdx.y];
    const T* S = base + mi.off + (long long)s_buf * mi.bufsz;
    T* Y = base + mi.off + (long long)y_buf * mi.bufsz;
    const float rho = st.rho_s[blockIdx.y];
    const float d = 2.f / rho, sc = 1.f / (rho * rho);
    const long long total = (long long)mi.n * mi.ld;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int r = (int)(idx / mi.ld), c = (int)(idx - (long long)r * mi.ld);
        float v = 0.f;
        if (c < mi.n) v = (r == c ? d : 0.f) - sc * Num<T>::to_f(S[idx]);
        Y[idx] = Num<T>::from_f(v);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) { st.inv_iters[blockIdx.y] = 1; st.ybuf[blockIdx.y] = y_buf; }
}

// ---------------------------------------------------------------------------------------------
// Plain FFMA grouped GEMM with the same GemmOp semantics as the tcgen05 kernel.
// grid = (max tiles of 64 x 64, nmat); 256 threads, 4 x 4 outputs each.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) k_gemm_simt(GemmOp op, T* base) {
    const int m = blockIdx.y;
    if (!gate_open(op, m)) return;
    const MatInfo mi = op.mats[m];
    const int nt = (mi.n + 63) / 64;
    if ((int)blockIdx.x >= nt * nt) return;
    const int tm = blockIdx.x / nt, tn = blockIdx.x - tm * nt;
    const int a_buf = op.a_buf >= 0 ? op.a_buf : op.st.ybuf[m];
    const T* A = base + mi.off + (long long)a_buf * mi.bufsz;
    const T* B = base + mi.off + (long long)op.b_buf * mi.bufsz;
    T* C = base + mi.off + (long long)op.c_buf * mi.bufsz;
    __shared__ float sA[16][64 + 4];
    __shared__ float sB[16][64 + 4];
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    float acc[4][4] = {};
    for (int k0 = 0; k0 < mi.n; k0 += 16) {
        for (int e = threadIdx.x; e < 64 * 16; e += 256) {
            const int r = e >> 4, k = e & 15;                  // A tile: 64 rows x 16 k
            const int gr = tm * 64 + r, gk = k0 + k;
            sA[k][r] = (gr < mi.n && gk < mi.n) ? Num<T>::to_f(A[(long long)gr * mi.ld + gk]) : 0.f;
            const int kb = e >> 6, c = e & 63;                 // B tile: 16 k x 64 cols
            const int gkb = k0 + kb, gc = tn * 64 + c;
            sB[kb][c] = (gkb < mi.n && gc < mi.n) ? Num<T>::to_f(B[(long long)gkb * mi.ld + gc]) : 0.f;
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
    const float alpha = op.alpha_arr ? op.alpha_arr[m] : op.alpha;
    float rsum = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int r = tm * 64 + ty * 4 + i;
        if (r >= mi.n) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int c = tn * 64 + tx * 4 + j;
            if (c >= mi.n) continue;
            const float x = alpha * acc[i][j];
            const float delta = (r == c) ? 1.f : 0.f;
            if (op.want_res) { const float d = x - delta; rsum += d * d; }
            C[(long long)r * mi.ld + c] = Num<T>::from_f(op.sgn * x + op.beta * delta);
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
            if (t != 0.f) atomicAdd(&op.st.res_acc[m], t);
        }
        tile_finished(op, m, nt * nt);
    }
}

// ---------------------------------------------------------------------------------------------
// a6 + a7: D_sub[:, cols(i)] = 1/2 (Y[:, cols] - X Y[:, cols])   (Eq. 8 with sign(A) = X, S^-1 = Y),
// scattered into slot (i, j) of the output as (D_ji)^T, and
// e_i = sum_j <D_ji, H0_ji> accumulated in FP64 (Eq. 4, H0 symmetric).
// grid = (row chunks, nmat); dynamic smem: float Yc[n][nbi], int off[cnt + 1].
// ---------------------------------------------------------------------------------------------
template <typename T, typename TV, typename TD>
__global__ void __launch_bounds__(256) k_dcols_scatter(SysView sv, const MatInfo* mats, BatchState st, const T* base,
                                                       const TV* H_vals, TD* D_vals, double* e_atom, int max_nset) {
    extern __shared__ unsigned char sm_raw[];
    const int m = blockIdx.y;
    const MatInfo mi = mats[m];
    if (st.status[m] & ST_NOTSPD) return;
    int* s_off = reinterpret_cast<int*>(sm_raw);                         // [max_nset + 1]
    float* s_y = reinterpret_cast<float*>(s_off + max_nset + 1);        // [n][nbi]
    const T* X = base + mi.off + (long long)st.xbuf[m] * mi.bufsz;
    const T* Y = base + mi.off + (long long)st.ybuf[m] * mi.bufsz;
    const long long p0 = sv.nset_ptr[mi.atom];
    const int cnt = (int)(sv.nset_ptr[mi.atom + 1] - p0);
    const int nbi = mi.nbi;
    for (int b = threadIdx.x; b < cnt; b += blockDim.x) s_off[b] = sv.nset_off[p0 + b];
    if (threadIdx.x == 0) s_off[cnt] = mi.n;
    for (int idx = threadIdx.x; idx < mi.n * nbi; idx += blockDim.x) {
        const int k = idx / nbi, c = idx - k * nbi;
        s_y[idx] = Num<T>::to_f(Y[(long long)k * mi.ld + mi.pos + c]);
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double e_part = 0.0;
    for (int r = blockIdx.x * 8 + warp; r < mi.n; r += gridDim.x * 8) {
        // which atom of N(i) owns row r (warp-uniform binary search)
        int lo = 0, hi = cnt - 1;
        while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (s_off[mid] <= r) lo = mid; else hi = mid - 1; }
        const int a = lo, bb = r - s_off[a], nbj = s_off[a + 1] - s_off[a];
        const long long out0 = sv.blk_off[sv.nset_slot[p0 + a]];
        const T* xrow = X + (long long)r * mi.ld;
        for (int c0 = 0; c0 < nbi; c0 += 16) {
            const int nc = min(16, nbi - c0);
            float acc[16];
#pragma unroll
            for (int c = 0; c < 16; ++c) acc[c] = 0.f;
            for (int k = lane; k < mi.n; k += 32) {
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
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e_part += __shfl_xor_sync(0xffffffffu, e_part, o);
    if (lane == 0 && e_part != 0.0) atomicAdd(&e_atom[mi.atom], e_part);
}

// per-atom statistics of a finished batch
__global__ void k_save_stats(const MatInfo* mats, BatchState st, int nmat, int* a_inv, int* a_sign, int* a_status,
                             int* a_gemms, float* a_res, float* a_rho) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= nmat) return;
    const int a = mats[m].atom;
    a_inv[a] = st.inv_iters[m]; a_sign[a] = st.sign_iters[m]; a_status[a] = st.status[m];
    a_gemms[a] = st.gemm_count[m]; a_res[a] = st.res_last[m]; a_rho[a] = st.rho_a[m];
}

// number of matrices for which phase (0 = inverse, 1 = sign) is still running
__global__ void k_count_active(BatchState st, int nmat, int phase, int* out) {
    __shared__ int cnt;
    if (threadIdx.x == 0) cnt = 0;
    __syncthreads();
    int c = 0;
    for (int m = threadIdx.x; m < nmat; m += blockDim.x) {
        if (phase == 0) c += st.inv_done[m] == 0;
        else c += (st.sign_done[m] == 0 && (st.status[m] & ST_NOTSPD) == 0);
    }
    if (c) atomicAdd(&cnt, c);
    __syncthreads();
    if (threadIdx.x == 0) *out = cnt;
}

// C-1 filter: keep[s] = max(|H0 block|_max, |S block|_max) > eps (diagonal handled on the host)
template <typename TV>
__global__ void k_block_keep(const long long* blk_off, const TV* H_vals, const TV* S_vals, long long nnzb, double eps,
                             unsigned char* keep) {
    const long long s = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (s >= nnzb) return;
    const int lane = threadIdx.x & 31;
    double mx = 0.0;
    for (long long e = blk_off[s] + lane; e < blk_off[s + 1]; e += 32)
        mx = fmax(mx, fmax(fabs((double)H_vals[e]), fabs((double)S_vals[e])));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (lane == 0) keep[s] = mx > eps ? 1 : 0;
}

}  // namespace nolsm
