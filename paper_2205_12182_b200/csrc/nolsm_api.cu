// C ABI of the NOLSM hot path (include/nolsm.h): context, assemble (a0), batch orchestration of the
// device pipeline (a1-a7) and diagnostics. Host code only plans and launches; every step of the path
// runs in the kernels of kernels.cuh and gemm_umma.cuh.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <thread>
#include <vector>

#include "../../include/nolsm.h"
#include "gemm_umma.cuh"
#include "kernels.cuh"
#include "tmap_host.h"

using namespace nolsm;

namespace {

struct Batch {
    int64_t first;   // index of the first matrix in the plan's MatInfo array
    int nmat;
    int ntiles;      // UMMA tiles (128 x bn)
    int max_tiles64; // max over matrices of ceil(n/64)^2 (SIMT grid)
    int max_n, max_ld, max_nset, max_nbi;
};

struct Plan {
    int64_t a0 = -1, a1 = -1;
    std::vector<Batch> batches;
    std::vector<MatInfo> mats;
    MatInfo* d_mats = nullptr;
    CUtensorMap* d_maps = nullptr;
};

template <typename F>
void parallel_for(int64_t n, F f) {
    unsigned nt = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
    if (n < 1 << 16) nt = 1;
    if (nt == 1) { f(0, n); return; }
    std::vector<std::thread> th;
    const int64_t chunk = (n + nt - 1) / nt;
    for (unsigned t = 0; t < nt; ++t) {
        const int64_t b = t * chunk, e = std::min<int64_t>(n, b + chunk);
        if (b < e) th.emplace_back([=] { f(b, e); });
    }
    for (auto& x : th) x.join();
}

}  // namespace

struct nolsm_ctx {
    int dev = 0;
    nolsm_options opt{};
    std::string err;
    bool assembled = false;
    int sms = 148;
    int tile_target = 0;

    // host copy of the pattern and derived index data
    int64_t n_atoms = 0, nnzb = 0, nvals = 0;
    std::vector<int32_t> atom_nb, col_idx, nset_atom, nset_slot, nset_off, dim, pos;
    std::vector<int64_t> row_ptr, blk_off, nset_ptr;
    bool filtered = false;

    // device arrays
    std::vector<void*> owned;           // everything cudaMalloc'ed by assemble (freed on re-assemble / destroy)
    long long *d_row_ptr = nullptr, *d_blk_off = nullptr, *d_nset_ptr = nullptr;
    int *d_col_idx = nullptr, *d_atom_nb = nullptr, *d_nset_atom = nullptr, *d_nset_slot = nullptr, *d_nset_off = nullptr;
    const void *dH = nullptr, *dS = nullptr;
    int val_dtype = NOLSM_DTYPE_F64;

    void* ws = nullptr;
    size_t ws_bytes = 0;
    int max_batch = 0;
    Plan plan;

    // batch state + per-atom results
    void* state_mem = nullptr;
    BatchState st{};
    float *d_vec = nullptr, *d_nrm = nullptr;
    int ldx = 0;
    int* d_flag = nullptr;
    int* h_flag = nullptr;
    int *a_inv = nullptr, *a_sign = nullptr, *a_status = nullptr, *a_gemms = nullptr;
    float *a_res = nullptr, *a_rho = nullptr;
    double* d_e_atom = nullptr;

    // last density call
    cudaStream_t last_stream = nullptr;
    int64_t last_a0 = 0, last_a1 = 0;
    bool have_result = false;
    void* d_D_stage = nullptr;
    size_t d_D_stage_bytes = 0;
    int inv_check_from = 3, sign_check_from = 6;
    double gather_bytes = 0, scatter_bytes = 0;
    size_t last_ds = 8;

    // sampled per-launch profiling (options.profile_every): CUDA events on the launching stream
    struct Rec { int kind; size_t ev; };
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    std::vector<Rec> recs;
    std::vector<std::pair<int64_t, int64_t>> prof_ranges;   // atom ranges of the sampled batches
    bool prof_on = false;
    double prof[NOLSM_PROFILE_LEN] = {};
    unsigned long long* d_gather_elems = nullptr;
    int64_t launches = 0;
};

enum { K_GATHER = 0, K_GEMM = 1, K_DCOLS = 2, K_OTHER = 3 };

namespace {

#define CU_TRY(ctx, expr)                                                                           \
    do {                                                                                            \
        cudaError_t e_ = (expr);                                                                    \
        if (e_ != cudaSuccess) {                                                                    \
            (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(e_);                       \
            return e_ == cudaErrorMemoryAllocation ? NOLSM_ENOMEM : NOLSM_ECUDA;                   \
        }                                                                                           \
    } while (0)

size_t prof_begin(nolsm_ctx* c, int kind, cudaStream_t s) {
    c->launches += 1;
    if (!c->prof_on) return 0;
    while (c->ev_pool.size() < c->ev_used + 2) {
        cudaEvent_t e;
        cudaEventCreate(&e);
        c->ev_pool.push_back(e);
    }
    const size_t i = c->ev_used;
    c->ev_used += 2;
    cudaEventRecord(c->ev_pool[i], s);
    c->recs.push_back({kind, i});
    return i;
}
void prof_end(nolsm_ctx* c, size_t i, cudaStream_t s) {
    if (c->prof_on) cudaEventRecord(c->ev_pool[i + 1], s);
}

#define LAUNCH(c, kind, s, ...)                      \
    do {                                             \
        const size_t pi_ = prof_begin(c, kind, s);   \
        __VA_ARGS__;                                 \
        prof_end(c, pi_, s);                         \
    } while (0)

int fail(nolsm_ctx* c, int code, const std::string& msg) {
    c->err = msg;
    return code;
}

bool is_device_ptr(const void* p) {
    cudaPointerAttributes at{};
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

int dmalloc(nolsm_ctx* c, void** p, size_t bytes) {
    CU_TRY(c, cudaMalloc(p, std::max<size_t>(bytes, 16)));
    c->owned.push_back(*p);
    return NOLSM_OK;
}

void free_assembled(nolsm_ctx* c) {
    for (void* p : c->owned) cudaFree(p);
    c->owned.clear();
    if (c->h_flag) { cudaFreeHost(c->h_flag); c->h_flag = nullptr; }
    if (c->d_D_stage) { cudaFree(c->d_D_stage); c->d_D_stage = nullptr; c->d_D_stage_bytes = 0; }
    c->ws = nullptr; c->plan = Plan(); c->assembled = false; c->have_result = false;
}

// Obtains a device view of a host-or-device array (copies host data into an owned buffer).
int to_device(nolsm_ctx* c, const void* src, size_t bytes, const void** out, cudaStream_t s) {
    if (is_device_ptr(src)) { *out = src; return NOLSM_OK; }
    void* d = nullptr;
    int r = dmalloc(c, &d, bytes);
    if (r) return r;
    CU_TRY(c, cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, s));
    *out = d;
    return NOLSM_OK;
}

int to_host(nolsm_ctx* c, const void* src, size_t bytes, void* dst, cudaStream_t s) {
    if (is_device_ptr(src)) {
        CU_TRY(c, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, s));
        CU_TRY(c, cudaStreamSynchronize(s));
    } else {
        memcpy(dst, src, bytes);
    }
    return NOLSM_OK;
}

size_t elem_size(const nolsm_ctx* c) { return c->opt.precision == NOLSM_PREC_FP32 ? 4 : 2; }
bool use_umma(const nolsm_ctx* c) {
    if (c->opt.precision == NOLSM_PREC_FP32) return false;
    return c->opt.gemm_backend != NOLSM_GEMM_SIMT;
}

void fill_matinfo(const nolsm_ctx* c, int64_t atom, MatInfo& mi) {
    const int n = c->dim[atom];
    mi.n = n;
    mi.ld = (n + 7) / 8 * 8;
    mi.pos = c->pos[atom];
    mi.nbi = c->atom_nb[atom];
    mi.ntn = (n + 255) / 256;
    int bn = ((n + mi.ntn - 1) / mi.ntn + 15) / 16 * 16;
    mi.bn = std::min(bn, 256);
    mi.ntn = (n + mi.bn - 1) / mi.bn;
    mi.atom = (int)atom;
    mi.bufsz = ((long long)n * mi.ld + 63) / 64 * 64;
    mi.tile_start = 0;
    mi.off = 0;
}

// Greedy batch plan over atoms [a0, a1): a batch is closed when it reaches the tile target, the
// matrix cap or the workspace capacity.
int build_plan(nolsm_ctx* c, int64_t a0, int64_t a1, cudaStream_t s) {
    Plan& p = c->plan;
    if (p.a0 == a0 && p.a1 == a1) return NOLSM_OK;
    if (p.d_mats) { cudaFree(p.d_mats); p.d_mats = nullptr; }
    if (p.d_maps) { cudaFree(p.d_maps); p.d_maps = nullptr; }
    p = Plan();
    p.mats.resize(a1 - a0);
    const size_t es = elem_size(c);
    Batch cur{};
    cur.first = 0;
    long long off = 0;
    auto close = [&]() { if (cur.nmat) { p.batches.push_back(cur); } };
    for (int64_t a = a0; a < a1; ++a) {
        MatInfo mi;
        fill_matinfo(c, a, mi);
        const long long need = mi.bufsz * NBUF;
        if ((size_t)(need * es) > c->ws_bytes) return fail(c, NOLSM_ENOMEM, "workspace too small for one submatrix");
        const bool full = cur.nmat > 0 && (cur.nmat >= c->max_batch || cur.ntiles >= c->tile_target ||
                                           (size_t)((off + need) * es) > c->ws_bytes);
        if (full) {
            close();
            cur = Batch{};
            cur.first = a - a0;
            off = 0;
        }
        mi.off = off;
        mi.tile_start = cur.ntiles;
        off += need;
        const int ntm = (mi.n + BM - 1) / BM;
        cur.ntiles += ntm * mi.ntn;
        const int t64 = (mi.n + 63) / 64;
        cur.max_tiles64 = std::max(cur.max_tiles64, t64 * t64);
        cur.max_n = std::max(cur.max_n, mi.n);
        cur.max_ld = std::max(cur.max_ld, mi.ld);
        cur.max_nset = std::max<int>(cur.max_nset, (int)(c->nset_ptr[a + 1] - c->nset_ptr[a]));
        cur.max_nbi = std::max(cur.max_nbi, mi.nbi);
        cur.nmat += 1;
        p.mats[a - a0] = mi;
    }
    close();
    CU_TRY(c, cudaMalloc((void**)&p.d_mats, std::max<size_t>(1, p.mats.size()) * sizeof(MatInfo)));
    CU_TRY(c, cudaMemcpyAsync(p.d_mats, p.mats.data(), p.mats.size() * sizeof(MatInfo), cudaMemcpyHostToDevice, s));
    if (use_umma(c)) {
        std::vector<CUtensorMap> maps(p.mats.size() * NBUF);
        std::atomic<bool> ok{true};
        if (!encode_tiled_fn()) return fail(c, NOLSM_ECUDA, "cuTensorMapEncodeTiled not available");
        parallel_for((int64_t)p.mats.size(), [&](int64_t b, int64_t e) {
            for (int64_t i = b; i < e; ++i) {
                const MatInfo& mi = p.mats[i];
                for (int k = 0; k < NBUF; ++k) {
                    const __half* base = (const __half*)c->ws + mi.off + (long long)k * mi.bufsz;
                    if (!make_tmap_f16_64x64(&maps[i * NBUF + k], base, mi.n, mi.ld)) ok = false;
                }
            }
        });
        if (!ok) return fail(c, NOLSM_ECUDA, "cuTensorMapEncodeTiled failed");
        CU_TRY(c, cudaMalloc((void**)&p.d_maps, std::max<size_t>(1, maps.size()) * sizeof(CUtensorMap)));
        CU_TRY(c, cudaMemcpyAsync(p.d_maps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, s));
        CU_TRY(c, cudaStreamSynchronize(s));   // `maps` is a local
    }
    p.a0 = a0;
    p.a1 = a1;
    return NOLSM_OK;
}

SysView sys_view(const nolsm_ctx* c) {
    SysView v;
    v.row_ptr = c->d_row_ptr; v.col_idx = c->d_col_idx; v.blk_off = c->d_blk_off; v.atom_nb = c->d_atom_nb;
    v.nset_ptr = c->d_nset_ptr; v.nset_atom = c->d_nset_atom; v.nset_slot = c->d_nset_slot; v.nset_off = c->d_nset_off;
    return v;
}

template <typename T>
int launch_gather(nolsm_ctx* c, const Batch& b, const MatInfo* d_mats, cudaStream_t s) {
    const size_t smem = (size_t)b.max_nset * 8 + (size_t)(b.max_nset + 1) * 4 + (size_t)b.max_ld * 2 + 16;
    dim3 grid(std::min(b.max_nset, 64), b.nmat, 2);
    if (c->val_dtype == NOLSM_DTYPE_F64) {
        auto k = k_gather<double, T>;
        CU_TRY(c, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(smem, 48 * 1024)));
        LAUNCH(c, K_GATHER, s, k<<<grid, 256, smem, s>>>(sys_view(c), d_mats, (const double*)c->dS, (const double*)c->dH, (T*)c->ws, b.max_nset, b.max_ld, c->prof_on ? c->d_gather_elems : nullptr));
    } else {
        auto k = k_gather<float, T>;
        CU_TRY(c, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(smem, 48 * 1024)));
        LAUNCH(c, K_GATHER, s, k<<<grid, 256, smem, s>>>(sys_view(c), d_mats, (const float*)c->dS, (const float*)c->dH, (T*)c->ws, b.max_nset, b.max_ld, c->prof_on ? c->d_gather_elems : nullptr));
    }
    CU_TRY(c, cudaGetLastError());
    return NOLSM_OK;
}

template <typename T>
int launch_gemm(nolsm_ctx* c, const Batch& b, GemmOp op, const CUtensorMap* d_maps, cudaStream_t s) {
    if (use_umma(c)) {
        UmmaArgs a;
        a.op = op;
        a.maps = d_maps;
        a.base = (__half*)c->ws;
        LAUNCH(c, K_GEMM, s, gemm_umma_kernel<<<std::min(c->sms, b.ntiles), UMMA_THREADS, UMMA_SMEM_BYTES, s>>>(a));
    } else {
        LAUNCH(c, K_GEMM, s, k_gemm_simt<T><<<dim3(b.max_tiles64, b.nmat), 256, 0, s>>>(op, (T*)c->ws));
    }
    CU_TRY(c, cudaGetLastError());
    return NOLSM_OK;
}

int count_active(nolsm_ctx* c, int nmat, int phase, cudaStream_t s, int* out) {
    LAUNCH(c, K_OTHER, s, k_count_active<<<1, 256, 0, s>>>(c->st, nmat, phase, c->d_flag));
    CU_TRY(c, cudaMemcpyAsync(c->h_flag, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, s));
    CU_TRY(c, cudaStreamSynchronize(s));
    *out = *c->h_flag;
    return NOLSM_OK;
}

template <typename T>
int power_iterations(nolsm_ctx* c, const Batch& b, const MatInfo* d_mats, int buf, int iters, int which, cudaStream_t s) {
    const int nm = b.nmat;
    CU_TRY(c, cudaMemsetAsync(c->d_nrm, 0, sizeof(float) * (size_t)(iters + 1) * c->max_batch, s));
    LAUNCH(c, K_OTHER, s, k_vec_init<<<dim3((b.max_n + 255) / 256, nm), 256, 0, s>>>(d_mats, c->d_vec, c->d_nrm, c->ldx));
    float* x = c->d_vec;
    float* y = c->d_vec + (size_t)c->max_batch * c->ldx;
    const int gx = std::max(1, std::min((b.max_n + 7) / 8, (4 * c->sms + nm - 1) / nm));
    for (int it = 0; it < iters; ++it) {
        LAUNCH(c, K_OTHER, s, k_matvec<T><<<dim3(gx, nm), 256, 0, s>>>(d_mats, (const T*)c->ws, buf, x, c->d_nrm + (size_t)it * c->max_batch, y,
                                                                      c->d_nrm + (size_t)(it + 1) * c->max_batch, c->ldx));
        std::swap(x, y);
    }
    LAUNCH(c, K_OTHER, s, k_rho_finish<<<(nm + 127) / 128, 128, 0, s>>>(c->st, c->d_nrm + (size_t)iters * c->max_batch, nm, which, 1.05f));
    CU_TRY(c, cudaGetLastError());
    return NOLSM_OK;
}

template <typename T, typename TD>
int launch_dcols(nolsm_ctx* c, const Batch& b, const MatInfo* d_mats, TD* D, cudaStream_t s) {
    const size_t smem = (size_t)(b.max_nset + 1) * 4 + (size_t)b.max_n * b.max_nbi * 4 + 16;
    const int gx = std::max(1, std::min((b.max_n + 7) / 8, (3 * c->sms + b.nmat - 1) / b.nmat));
    dim3 grid(gx, b.nmat);
    if (c->val_dtype == NOLSM_DTYPE_F64) {
        auto k = k_dcols_scatter<T, double, TD>;
        CU_TRY(c, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(smem, 48 * 1024)));
        LAUNCH(c, K_DCOLS, s, k<<<grid, 256, smem, s>>>(sys_view(c), d_mats, c->st, (const T*)c->ws, (const double*)c->dH, D, c->d_e_atom, b.max_nset));
    } else {
        auto k = k_dcols_scatter<T, float, TD>;
        CU_TRY(c, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(smem, 48 * 1024)));
        LAUNCH(c, K_DCOLS, s, k<<<grid, 256, smem, s>>>(sys_view(c), d_mats, c->st, (const T*)c->ws, (const float*)c->dH, D, c->d_e_atom, b.max_nset));
    }
    CU_TRY(c, cudaGetLastError());
    return NOLSM_OK;
}

// One batch through a1-a7.
template <typename T>
int run_batch(nolsm_ctx* c, const Batch& b, double mu, void* D, int d_dtype, cudaStream_t s) {
    const MatInfo* d_mats = c->plan.d_mats + b.first;
    const CUtensorMap* d_maps = c->plan.d_maps ? c->plan.d_maps + b.first * NBUF : nullptr;
    const int nm = b.nmat;
    int r;
    LAUNCH(c, K_OTHER, s, k_state_init<<<(nm + 127) / 128, 128, 0, s>>>(c->st, nm));
    if ((r = launch_gather<T>(c, b, d_mats, s))) return r;

    GemmOp op{};
    op.nmat = nm; op.ntiles = b.ntiles; op.mats = d_mats; op.st = c->st;
    op.alpha = 1.f; op.alpha_arr = nullptr;

    // ---- a2: S_sub^-1 by the Schulz iteration, Y0 = I / rho(S) ----
    if ((r = power_iterations<T>(c, b, d_mats, 0, c->opt.power_iters_s, 0, s))) return r;
    LAUNCH(c, K_OTHER, s, k_schulz_first<T><<<dim3(std::max(1, std::min(64, (b.max_n * b.max_ld + 2047) / 2048)), nm), 256, 0, s>>>(
                              d_mats, c->st, (T*)c->ws, 0, 2));
    int ran = 1;
    for (int k = 1; k < c->opt.max_inv_iters; ++k) {
        const int ycur = (k & 1) ? 2 : 3, ynext = 5 - ycur;
        op.a_buf = 0; op.b_buf = ycur; op.c_buf = 4; op.sgn = -1.f; op.beta = 2.f; op.want_res = 1;
        op.alpha = 1.f; op.alpha_arr = nullptr;
        op.gate = GATE_INV_ACTIVE; op.finish = FIN_INV_G1; op.tol = c->opt.tol_inv; op.max_iters = c->opt.max_inv_iters;
        if ((r = launch_gemm<T>(c, b, op, d_maps, s))) return r;
        op.a_buf = ycur; op.b_buf = 4; op.c_buf = ynext; op.sgn = 1.f; op.beta = 0.f; op.want_res = 0;
        op.finish = FIN_INV_G2;
        if ((r = launch_gemm<T>(c, b, op, d_maps, s))) return r;
        ran = k + 1;
        if (k + 1 >= c->inv_check_from) {
            int active;
            if ((r = count_active(c, nm, 0, s, &active))) return r;
            if (!active) break;
        }
    }
    c->inv_check_from = std::max(2, ran - 1);

    // ---- a3: A = S^-1 H - mu I (into buffer 0), rho(A) ----
    op.a_buf = -1; op.b_buf = 1; op.c_buf = 0; op.sgn = 1.f; op.beta = (float)(-mu); op.want_res = 0;
    op.alpha = 1.f; op.alpha_arr = nullptr; op.gate = GATE_INV_OK; op.finish = FIN_COUNT_ONLY;
    if ((r = launch_gemm<T>(c, b, op, d_maps, s))) return r;
    if ((r = power_iterations<T>(c, b, d_mats, 0, c->opt.power_iters_a, 1, s))) return r;

    // ---- a4 + a5: Newton-Schulz sign iteration (Eq. 6) with fused residual ----
    ran = 0;
    for (int k = 0; k < c->opt.max_sign_iters; ++k) {
        const int xcur = k & 1, xnext = 1 - xcur;
        op.a_buf = xcur; op.b_buf = xcur; op.c_buf = 4; op.sgn = -1.f; op.beta = 3.f; op.want_res = 1;
        op.alpha = 1.f; op.alpha_arr = k == 0 ? c->st.alpha1 : nullptr;
        op.gate = GATE_SIGN_ACTIVE; op.finish = FIN_SIGN_G1; op.tol = c->opt.tol_sign; op.max_iters = c->opt.max_sign_iters;
        if ((r = launch_gemm<T>(c, b, op, d_maps, s))) return r;
        op.a_buf = xcur; op.b_buf = 4; op.c_buf = xnext; op.sgn = 1.f; op.beta = 0.f; op.want_res = 0;
        op.alpha = 0.5f; op.alpha_arr = k == 0 ? c->st.alpha2 : nullptr;
        op.finish = FIN_SIGN_G2;
        if ((r = launch_gemm<T>(c, b, op, d_maps, s))) return r;
        ran = k + 1;
        if (k + 1 >= c->sign_check_from) {
            int active;
            if ((r = count_active(c, nm, 1, s, &active))) return r;
            if (!active) break;
        }
    }
    c->sign_check_from = std::max(2, ran - 1);

    // ---- a6 + a7: D columns, scatter, energy partials ----
    if (d_dtype == NOLSM_DTYPE_F64) r = launch_dcols<T, double>(c, b, d_mats, (double*)D, s);
    else r = launch_dcols<T, float>(c, b, d_mats, (float*)D, s);
    if (r) return r;
    LAUNCH(c, K_OTHER, s, k_save_stats<<<(nm + 127) / 128, 128, 0, s>>>(d_mats, c->st, nm, c->a_inv, c->a_sign, c->a_status,
                                                                        c->a_gemms, c->a_res, c->a_rho));
    CU_TRY(c, cudaGetLastError());
    return NOLSM_OK;
}

int getenv_int(const char* name, int dflt) {
    const char* v = getenv(name);
    return v && *v ? atoi(v) : dflt;
}

}  // namespace

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

int nolsm_create(nolsm_ctx** out, int cuda_device, const nolsm_options* opt) {
    if (!out) return NOLSM_EINVAL;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) {
        cudaGetLastError();
        return NOLSM_ECUDA;
    }
    nolsm_ctx* c = new (std::nothrow) nolsm_ctx();
    if (!c) return NOLSM_ENOMEM;
    c->dev = cuda_device;
    if (opt) c->opt = *opt;
    nolsm_options& o = c->opt;
    const bool fp32 = o.precision == NOLSM_PREC_FP32;
    if (o.precision != NOLSM_PREC_FP16_FP32 && !fp32) { delete c; return NOLSM_EINVAL; }
    if (o.max_inv_iters <= 0) o.max_inv_iters = 24;
    if (o.max_sign_iters <= 0) o.max_sign_iters = 64;
    if (o.tol_inv <= 0) o.tol_inv = fp32 ? 1e-5f : 2e-3f;
    if (o.tol_sign <= 0) o.tol_sign = fp32 ? 1e-5f : 2e-3f;
    if (o.power_iters_s <= 0) o.power_iters_s = 6;
    if (o.power_iters_a <= 0) o.power_iters_a = 12;
    if (o.eps_filter < 0) { delete c; return NOLSM_EINVAL; }
    cudaSetDevice(cuda_device);
    cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, cuda_device);
    if (getenv_int("NOLSM_PROFILE_EVERY", 0) > 0) o.profile_every = getenv_int("NOLSM_PROFILE_EVERY", 0);
    c->tile_target = getenv_int("NOLSM_BATCH_TILES", 8 * c->sms);
    if (use_umma(c)) {
        if (cudaFuncSetAttribute(gemm_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, UMMA_SMEM_BYTES) != cudaSuccess) {
            cudaGetLastError();
            delete c;
            return NOLSM_ECUDA;
        }
    }
    *out = c;
    return NOLSM_OK;
}

int nolsm_destroy(nolsm_ctx* c) {
    if (!c) return NOLSM_EINVAL;
    cudaSetDevice(c->dev);
    if (c->plan.d_mats) cudaFree(c->plan.d_mats);
    if (c->plan.d_maps) cudaFree(c->plan.d_maps);
    c->plan.d_mats = nullptr; c->plan.d_maps = nullptr;
    free_assembled(c);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    delete c;
    return NOLSM_OK;
}

const char* nolsm_last_error(const nolsm_ctx* c) { return c ? c->err.c_str() : "null context"; }

int nolsm_assemble(nolsm_ctx* c, int64_t n_atoms, const int32_t* atom_nb, const int64_t* row_ptr,
                   const int32_t* col_idx, const void* H0_vals, const void* S_vals, int val_dtype, void* cuda_stream) {
    if (!c) return NOLSM_EINVAL;
    if (n_atoms <= 0 || !atom_nb || !row_ptr || !col_idx || !H0_vals || !S_vals)
        return fail(c, NOLSM_EINVAL, "null pointer or n_atoms <= 0");
    if (val_dtype != NOLSM_DTYPE_F64 && val_dtype != NOLSM_DTYPE_F32) return fail(c, NOLSM_EINVAL, "bad val_dtype");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaSetDevice(c->dev);
    if (c->plan.d_mats) { cudaFree(c->plan.d_mats); c->plan.d_mats = nullptr; }
    if (c->plan.d_maps) { cudaFree(c->plan.d_maps); c->plan.d_maps = nullptr; }
    free_assembled(c);
    int r;
    c->n_atoms = n_atoms;
    c->val_dtype = val_dtype;
    c->atom_nb.resize(n_atoms);
    c->row_ptr.resize(n_atoms + 1);
    if ((r = to_host(c, atom_nb, sizeof(int32_t) * n_atoms, c->atom_nb.data(), s))) return r;
    if ((r = to_host(c, row_ptr, sizeof(int64_t) * (n_atoms + 1), c->row_ptr.data(), s))) return r;
    if (c->row_ptr[0] != 0) return fail(c, NOLSM_EINVAL, "row_ptr[0] != 0");
    for (int64_t i = 0; i < n_atoms; ++i) {
        if (c->atom_nb[i] <= 0) return fail(c, NOLSM_EINVAL, "atom_nb <= 0");
        if (c->row_ptr[i + 1] < c->row_ptr[i]) return fail(c, NOLSM_EINVAL, "row_ptr not monotone");
    }
    c->nnzb = c->row_ptr[n_atoms];
    if (c->nnzb <= 0 || c->nnzb >= (1ll << 31)) return fail(c, NOLSM_EINVAL, "nnzb out of range");
    c->col_idx.resize(c->nnzb);
    if ((r = to_host(c, col_idx, sizeof(int32_t) * c->nnzb, c->col_idx.data(), s))) return r;

    // ---- validation: ascending columns, diagonal present, structurally symmetric (C-5) ----
    std::atomic<int> bad{0};
    parallel_for(n_atoms, [&](int64_t b, int64_t e) {
        for (int64_t i = b; i < e && !bad; ++i) {
            bool diag = false;
            for (int64_t p = c->row_ptr[i]; p < c->row_ptr[i + 1]; ++p) {
                const int64_t j = c->col_idx[p];
                if (j < 0 || j >= n_atoms) { bad = 1; break; }
                if (p > c->row_ptr[i] && c->col_idx[p - 1] >= j) { bad = 2; break; }
                if (j == i) diag = true;
                else {
                    const int32_t* lo = c->col_idx.data() + c->row_ptr[j];
                    const int32_t* hi = c->col_idx.data() + c->row_ptr[j + 1];
                    const int32_t* it = std::lower_bound(lo, hi, (int32_t)i);
                    if (it == hi || *it != i) { bad = 3; break; }
                }
            }
            if (!bad && !diag) bad = 4;
        }
    });
    if (bad) {
        static const char* why[] = {"", "column index out of range", "columns not strictly ascending",
                                    "pattern not structurally symmetric", "diagonal block missing"};
        return fail(c, NOLSM_EINVAL, why[bad.load()]);
    }

    // ---- block offsets ----
    c->blk_off.resize(c->nnzb + 1);
    c->blk_off[0] = 0;
    for (int64_t i = 0; i < n_atoms; ++i)
        for (int64_t p = c->row_ptr[i]; p < c->row_ptr[i + 1]; ++p)
            c->blk_off[p + 1] = c->blk_off[p] + (int64_t)c->atom_nb[i] * c->atom_nb[c->col_idx[p]];
    c->nvals = c->blk_off[c->nnzb];
    const size_t vs = val_dtype == NOLSM_DTYPE_F64 ? 8 : 4;

    // ---- device copies of pattern and values ----
    const void* tmp;
    if ((r = to_device(c, c->row_ptr.data(), sizeof(int64_t) * (n_atoms + 1), &tmp, s))) return r;
    c->d_row_ptr = (long long*)tmp;
    if ((r = to_device(c, c->col_idx.data(), sizeof(int32_t) * c->nnzb, &tmp, s))) return r;
    c->d_col_idx = (int*)tmp;
    if ((r = to_device(c, c->atom_nb.data(), sizeof(int32_t) * n_atoms, &tmp, s))) return r;
    c->d_atom_nb = (int*)tmp;
    if ((r = to_device(c, c->blk_off.data(), sizeof(int64_t) * (c->nnzb + 1), &tmp, s))) return r;
    c->d_blk_off = (long long*)tmp;
    if ((r = to_device(c, H0_vals, vs * c->nvals, &c->dH, s))) return r;
    if ((r = to_device(c, S_vals, vs * c->nvals, &c->dS, s))) return r;

    // ---- index sets N(i) (C-1 filter) ----
    std::vector<unsigned char> keep;
    c->filtered = c->opt.eps_filter > 0;
    if (c->filtered) {
        unsigned char* d_keep;
        if ((r = dmalloc(c, (void**)&d_keep, c->nnzb))) return r;
        const int wpb = 8;
        const unsigned grid = (unsigned)((c->nnzb + wpb - 1) / wpb);
        if (val_dtype == NOLSM_DTYPE_F64)
            k_block_keep<double><<<grid, wpb * 32, 0, s>>>(c->d_blk_off, (const double*)c->dH, (const double*)c->dS, c->nnzb, c->opt.eps_filter, d_keep);
        else
            k_block_keep<float><<<grid, wpb * 32, 0, s>>>(c->d_blk_off, (const float*)c->dH, (const float*)c->dS, c->nnzb, c->opt.eps_filter, d_keep);
        keep.resize(c->nnzb);
        CU_TRY(c, cudaMemcpyAsync(keep.data(), d_keep, c->nnzb, cudaMemcpyDeviceToHost, s));
        CU_TRY(c, cudaStreamSynchronize(s));
    }
    c->nset_ptr.assign(n_atoms + 1, 0);
    for (int64_t i = 0; i < n_atoms; ++i) {
        int64_t cnt = 0;
        for (int64_t p = c->row_ptr[i]; p < c->row_ptr[i + 1]; ++p)
            cnt += (!c->filtered || keep[p] || c->col_idx[p] == i) ? 1 : 0;
        c->nset_ptr[i + 1] = c->nset_ptr[i] + cnt;
    }
    const int64_t nn = c->nset_ptr[n_atoms];
    c->nset_atom.resize(nn); c->nset_slot.resize(nn); c->nset_off.resize(nn);
    c->dim.resize(n_atoms); c->pos.resize(n_atoms);
    parallel_for(n_atoms, [&](int64_t b, int64_t e) {
        for (int64_t i = b; i < e; ++i) {
            int64_t q = c->nset_ptr[i];
            int off = 0;
            for (int64_t p = c->row_ptr[i]; p < c->row_ptr[i + 1]; ++p) {
                const int32_t j = c->col_idx[p];
                if (c->filtered && !keep[p] && j != i) continue;
                c->nset_atom[q] = j; c->nset_slot[q] = (int32_t)p; c->nset_off[q] = off;
                if (j == i) c->pos[i] = off;
                off += c->atom_nb[j];
                ++q;
            }
            c->dim[i] = off;
        }
    });
    int max_n = 0;
    for (int64_t i = 0; i < n_atoms; ++i) max_n = std::max(max_n, c->dim[i]);
    if (max_n > 65535) return fail(c, NOLSM_EINVAL, "submatrix dimension > 65535 not supported");
    if (!c->filtered) {
        c->d_nset_ptr = c->d_row_ptr;
        c->d_nset_atom = c->d_col_idx;
    } else {
        if ((r = to_device(c, c->nset_ptr.data(), sizeof(int64_t) * (n_atoms + 1), &tmp, s))) return r;
        c->d_nset_ptr = (long long*)tmp;
        if ((r = to_device(c, c->nset_atom.data(), sizeof(int32_t) * nn, &tmp, s))) return r;
        c->d_nset_atom = (int*)tmp;
    }
    if ((r = to_device(c, c->nset_slot.data(), sizeof(int32_t) * nn, &tmp, s))) return r;
    c->d_nset_slot = (int*)tmp;
    if ((r = to_device(c, c->nset_off.data(), sizeof(int32_t) * nn, &tmp, s))) return r;
    c->d_nset_off = (int*)tmp;

    // ---- workspace, batch capacity, state ----
    const size_t es = elem_size(c);
    const long long max_ld = (max_n + 7) / 8 * 8;
    const size_t one = (size_t)(((long long)max_n * max_ld + 63) / 64 * 64) * NBUF * es;
    size_t free_b = 0, total_b = 0;
    CU_TRY(c, cudaMemGetInfo(&free_b, &total_b));
    // enough slots of the largest matrix to reach the tile target, within the caps
    const int tiles_one = std::max(1, ((max_n + BM - 1) / BM) * ((max_n + 255) / 256));
    size_t want = one * (size_t)std::max(2, (c->tile_target + tiles_one - 1) / tiles_one + 1) * 2;
    size_t cap = c->opt.workspace_bytes ? c->opt.workspace_bytes : std::min<size_t>(free_b / 2, (size_t)32 << 30);
    c->ws_bytes = std::max(one, std::min(want, cap));
    if ((r = dmalloc(c, &c->ws, c->ws_bytes))) return r;
    c->max_batch = c->opt.batch_atoms > 0 ? c->opt.batch_atoms : 4096;
    // smallest matrix bounds how many fit
    int min_n = max_n;
    for (int64_t i = 0; i < n_atoms; ++i) min_n = std::min(min_n, c->dim[i]);
    const size_t smallest = (size_t)(((long long)min_n * ((min_n + 7) / 8 * 8) + 63) / 64 * 64) * NBUF * es;
    c->max_batch = (int)std::min<size_t>(c->max_batch, std::max<size_t>(1, c->ws_bytes / smallest));
    c->max_batch = (int)std::min<int64_t>(c->max_batch, n_atoms);
    const int mb = c->max_batch;
    {
        const size_t nf = 7, ni = 11;
        if ((r = dmalloc(c, &c->state_mem, (nf * 4 + ni * 4) * (size_t)mb))) return r;
        float* f = (float*)c->state_mem;
        int* ii = (int*)(f + nf * mb);
        BatchState& st = c->st;
        st.res_acc = f; st.res_prev = f + mb; st.res_last = f + 2 * mb; st.rho_s = f + 3 * mb; st.rho_a = f + 4 * mb;
        st.alpha1 = f + 5 * mb; st.alpha2 = f + 6 * mb;
        st.tiles_done = ii; st.inv_conv = ii + mb; st.inv_done = ii + 2 * mb; st.inv_iters = ii + 3 * mb; st.ybuf = ii + 4 * mb;
        st.sign_conv = ii + 5 * mb; st.sign_done = ii + 6 * mb; st.sign_iters = ii + 7 * mb; st.xbuf = ii + 8 * mb;
        st.status = ii + 9 * mb; st.gemm_count = ii + 10 * mb;
    }
    c->ldx = (int)max_ld;
    const int pit = std::max(c->opt.power_iters_s, c->opt.power_iters_a) + 1;
    if ((r = dmalloc(c, (void**)&c->d_vec, sizeof(float) * 2 * (size_t)mb * c->ldx))) return r;
    if ((r = dmalloc(c, (void**)&c->d_nrm, sizeof(float) * (size_t)pit * mb))) return r;
    if ((r = dmalloc(c, (void**)&c->d_flag, 16))) return r;
    if ((r = dmalloc(c, (void**)&c->d_gather_elems, 16))) return r;
    CU_TRY(c, cudaMallocHost((void**)&c->h_flag, 16));
    if ((r = dmalloc(c, (void**)&c->a_inv, 4 * n_atoms))) return r;
    if ((r = dmalloc(c, (void**)&c->a_sign, 4 * n_atoms))) return r;
    if ((r = dmalloc(c, (void**)&c->a_status, 4 * n_atoms))) return r;
    if ((r = dmalloc(c, (void**)&c->a_gemms, 4 * n_atoms))) return r;
    if ((r = dmalloc(c, (void**)&c->a_res, 4 * n_atoms))) return r;
    if ((r = dmalloc(c, (void**)&c->a_rho, 4 * n_atoms))) return r;
    if ((r = dmalloc(c, (void**)&c->d_e_atom, 8 * n_atoms))) return r;
    CU_TRY(c, cudaMemsetAsync(c->a_inv, 0, 4 * n_atoms, s));
    CU_TRY(c, cudaMemsetAsync(c->a_sign, 0, 4 * n_atoms, s));
    CU_TRY(c, cudaMemsetAsync(c->a_status, 0, 4 * n_atoms, s));
    CU_TRY(c, cudaMemsetAsync(c->a_gemms, 0, 4 * n_atoms, s));
    CU_TRY(c, cudaMemsetAsync(c->a_res, 0, 4 * n_atoms, s));
    CU_TRY(c, cudaMemsetAsync(c->d_e_atom, 0, 8 * n_atoms, s));
    c->assembled = true;   // build_plan needs the workspace pointer
    if ((r = build_plan(c, 0, n_atoms, s))) { c->assembled = false; return r; }
    CU_TRY(c, cudaStreamSynchronize(s));
    return NOLSM_OK;
}

int nolsm_density_matrix_range(nolsm_ctx* c, double mu, int64_t a0, int64_t a1, void* D_vals, int d_dtype,
                               double* e_partial_host, void* cuda_stream) {
    if (!c) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "nolsm_assemble has not been called");
    if (!D_vals || a0 < 0 || a1 > c->n_atoms || a0 >= a1) return fail(c, NOLSM_EINVAL, "bad range or null D_vals");
    if (d_dtype != NOLSM_DTYPE_F64 && d_dtype != NOLSM_DTYPE_F32) return fail(c, NOLSM_EINVAL, "bad d_dtype");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaSetDevice(c->dev);
    int r;
    if ((r = build_plan(c, a0, a1, s))) return r;
    const size_t ds = d_dtype == NOLSM_DTYPE_F64 ? 8 : 4;
    c->last_ds = ds;
    const int64_t v0 = c->blk_off[c->row_ptr[a0]], v1 = c->blk_off[c->row_ptr[a1]];
    // device view of the output rows [a0, a1): D_dev points at element 0 of the whole array
    char* D_dev;
    const bool host_out = !is_device_ptr(D_vals);
    if (host_out) {
        const size_t need = (size_t)(v1 - v0) * ds;
        if (c->d_D_stage_bytes < need) {
            if (c->d_D_stage) cudaFree(c->d_D_stage);
            c->d_D_stage = nullptr; c->d_D_stage_bytes = 0;
            CU_TRY(c, cudaMalloc(&c->d_D_stage, need));
            c->d_D_stage_bytes = need;
        }
        D_dev = (char*)c->d_D_stage - (size_t)v0 * ds;
    } else {
        D_dev = (char*)D_vals;
    }
    CU_TRY(c, cudaMemsetAsync(D_dev + (size_t)v0 * ds, 0, (size_t)(v1 - v0) * ds, s));
    CU_TRY(c, cudaMemsetAsync(c->d_e_atom + a0, 0, 8 * (a1 - a0), s));
    c->gather_bytes = 0; c->scatter_bytes = 0;
    c->ev_used = 0; c->recs.clear(); c->prof_ranges.clear(); c->launches = 0;
    CU_TRY(c, cudaMemsetAsync(c->d_gather_elems, 0, 8, s));
    int64_t bi = 0;
    for (const Batch& b : c->plan.batches) {
        c->prof_on = c->opt.profile_every > 0 && (bi++ % c->opt.profile_every) == 0;
        if (c->prof_on) c->prof_ranges.push_back({a0 + b.first, a0 + b.first + b.nmat});
        r = c->opt.precision == NOLSM_PREC_FP32 ? run_batch<float>(c, b, mu, D_dev, d_dtype, s)
                                                : run_batch<__half>(c, b, mu, D_dev, d_dtype, s);
        c->prof_on = false;
        if (r) return r;
    }
    const size_t es = elem_size(c);
    const size_t vs = c->val_dtype == NOLSM_DTYPE_F64 ? 8 : 4;
    for (int64_t a = a0; a < a1; ++a) {
        const double n = c->dim[a], ld = (c->dim[a] + 7) / 8 * 8;
        const double nv = (double)(c->blk_off[c->row_ptr[a + 1]] - c->blk_off[c->row_ptr[a]]);
        c->gather_bytes += 2.0 * n * ld * es;                    // dense S_sub and H_sub written
        c->scatter_bytes += nv * (ds + vs) + 2.0 * n * ld * es;  // D row written, H0 row read, X and Y columns read
    }
    if (host_out) CU_TRY(c, cudaMemcpyAsync((char*)D_vals + (size_t)v0 * ds, c->d_D_stage, (size_t)(v1 - v0) * ds, cudaMemcpyDeviceToHost, s));
    c->last_stream = s; c->last_a0 = a0; c->last_a1 = a1; c->have_result = true;
    if (e_partial_host) return nolsm_energy(c, e_partial_host);
    return NOLSM_OK;
}

int nolsm_density_matrix(nolsm_ctx* c, double mu, void* D_vals, int d_dtype, void* cuda_stream) {
    if (!c) return NOLSM_EINVAL;
    return nolsm_density_matrix_range(c, mu, 0, c->n_atoms, D_vals, d_dtype, nullptr, cuda_stream);
}

int nolsm_energy(nolsm_ctx* c, double* e_elec) {
    if (!c || !e_elec) return NOLSM_EINVAL;
    if (!c->have_result) return fail(c, NOLSM_ESTATE, "no density matrix has been computed");
    cudaSetDevice(c->dev);
    CU_TRY(c, cudaStreamSynchronize(c->last_stream));
    const int64_t n = c->last_a1 - c->last_a0;
    std::vector<double> e(n);
    std::vector<int> st(n);
    CU_TRY(c, cudaMemcpy(e.data(), c->d_e_atom + c->last_a0, 8 * n, cudaMemcpyDeviceToHost));
    CU_TRY(c, cudaMemcpy(st.data(), c->a_status + c->last_a0, 4 * n, cudaMemcpyDeviceToHost));
    double sum = 0;
    int bits = 0;
    for (int64_t i = 0; i < n; ++i) { sum += e[i]; bits |= st[i]; }
    *e_elec = sum;
    if (bits & ST_NOTSPD) return fail(c, NOLSM_ENOTSPD, "an S_sub inverse iteration failed (see nolsm_get_atom_stats)");
    if (bits & ST_NOCONV) return fail(c, NOLSM_ENOCONV, "a sign iteration hit max_sign_iters (see nolsm_get_atom_stats)");
    return NOLSM_OK;
}

int nolsm_get_index_set(nolsm_ctx* c, int64_t atom, int32_t* atoms_out, int32_t* n_inout, int32_t* dim_out) {
    if (!c || !n_inout) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    if (atom < 0 || atom >= c->n_atoms) return fail(c, NOLSM_EINVAL, "atom out of range");
    const int64_t p0 = c->nset_ptr[atom], cnt = c->nset_ptr[atom + 1] - p0;
    if (dim_out) *dim_out = c->dim[atom];
    if (atoms_out) {
        if (*n_inout < cnt) { *n_inout = (int32_t)cnt; return fail(c, NOLSM_EINVAL, "atoms_out too small"); }
        memcpy(atoms_out, c->nset_atom.data() + p0, sizeof(int32_t) * cnt);
    }
    *n_inout = (int32_t)cnt;
    return NOLSM_OK;
}

int nolsm_gather_submatrix(nolsm_ctx* c, int64_t atom, int which, int out_fp16, void* out_host) {
    if (!c || !out_host || (which != 0 && which != 1)) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    if (atom < 0 || atom >= c->n_atoms) return fail(c, NOLSM_EINVAL, "atom out of range");
    cudaSetDevice(c->dev);
    MatInfo mi;
    fill_matinfo(c, atom, mi);
    Batch b{};
    b.first = 0; b.nmat = 1; b.max_n = mi.n; b.max_ld = mi.ld; b.max_nbi = mi.nbi;
    b.max_nset = (int)(c->nset_ptr[atom + 1] - c->nset_ptr[atom]);
    MatInfo* d_mi;
    CU_TRY(c, cudaMalloc((void**)&d_mi, sizeof(MatInfo)));
    CU_TRY(c, cudaMemcpy(d_mi, &mi, sizeof(MatInfo), cudaMemcpyHostToDevice));
    int r = out_fp16 ? launch_gather<__half>(c, b, d_mi, nullptr) : launch_gather<float>(c, b, d_mi, nullptr);
    const size_t es = out_fp16 ? 2 : 4;
    if (!r) {
        cudaError_t e = cudaMemcpy2D(out_host, (size_t)mi.n * es, (const char*)c->ws + (size_t)which * mi.bufsz * es,
                                     (size_t)mi.ld * es, (size_t)mi.n * es, mi.n, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { c->err = cudaGetErrorString(e); r = NOLSM_ECUDA; }
    }
    cudaFree(d_mi);
    return r;
}

int nolsm_get_atom_stats(nolsm_ctx* c, int64_t a0, int64_t count, int32_t* dims, int32_t* inv_iters, int32_t* sign_iters,
                         int32_t* status, int32_t* gemms, float* residual, double* e_atom) {
    if (!c) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    if (a0 < 0 || count < 0 || a0 + count > c->n_atoms) return fail(c, NOLSM_EINVAL, "range");
    cudaSetDevice(c->dev);
    if (c->have_result) CU_TRY(c, cudaStreamSynchronize(c->last_stream));
    if (dims) memcpy(dims, c->dim.data() + a0, 4 * count);
    if (inv_iters) CU_TRY(c, cudaMemcpy(inv_iters, c->a_inv + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (sign_iters) CU_TRY(c, cudaMemcpy(sign_iters, c->a_sign + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (status) CU_TRY(c, cudaMemcpy(status, c->a_status + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (gemms) CU_TRY(c, cudaMemcpy(gemms, c->a_gemms + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (residual) CU_TRY(c, cudaMemcpy(residual, c->a_res + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (e_atom) CU_TRY(c, cudaMemcpy(e_atom, c->d_e_atom + a0, 8 * count, cudaMemcpyDeviceToHost));
    return NOLSM_OK;
}

int nolsm_get_stats(nolsm_ctx* c, nolsm_stats* out) {
    if (!c || !out) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    memset(out, 0, sizeof(*out));
    const int64_t n = c->n_atoms;
    out->n_atoms = n;
    out->n_batches = (int64_t)c->plan.batches.size();
    out->dim_min = 1 << 30;
    double dsum = 0;
    for (int64_t i = 0; i < n; ++i) {
        out->dim_min = std::min<int64_t>(out->dim_min, c->dim[i]);
        out->dim_max = std::max<int64_t>(out->dim_max, c->dim[i]);
        dsum += c->dim[i];
    }
    out->dim_mean = dsum / n;
    if (c->have_result) {
        std::vector<int32_t> inv(n), sg(n), st(n), gm(n);
        int r = nolsm_get_atom_stats(c, 0, n, nullptr, inv.data(), sg.data(), st.data(), gm.data(), nullptr, nullptr);
        if (r) return r;
        for (int64_t i = c->last_a0; i < c->last_a1; ++i) {
            out->sum_inv_iters += inv[i]; out->sum_sign_iters += sg[i]; out->gemms_executed += gm[i];
            const double d = c->dim[i];
            out->flops_useful += 2.0 * d * d * d * gm[i];
            MatInfo mi;
            fill_matinfo(c, i, mi);
            const double pm = (double)((mi.n + BM - 1) / BM) * BM, pn = (double)mi.ntn * mi.bn, pk = (double)((mi.n + 15) / 16) * 16;
            out->flops_padded += 2.0 * pm * pn * pk * gm[i];
            out->n_notspd += (st[i] & ST_NOTSPD) ? 1 : 0;
            out->n_noconv += (st[i] & ST_NOCONV) ? 1 : 0;
        }
        out->gather_bytes = c->gather_bytes;
        out->scatter_bytes = c->scatter_bytes;
    }
    return NOLSM_OK;
}

int nolsm_get_profile(nolsm_ctx* c, double* out, int n) {
    if (!c || !out || n < NOLSM_PROFILE_LEN) return NOLSM_EINVAL;
    if (!c->have_result) return fail(c, NOLSM_ESTATE, "no density matrix has been computed");
    cudaSetDevice(c->dev);
    CU_TRY(c, cudaStreamSynchronize(c->last_stream));
    double ms[4] = {0, 0, 0, 0}, cnt[4] = {0, 0, 0, 0};
    for (const nolsm_ctx::Rec& r : c->recs) {
        float t = 0;
        if (cudaEventElapsedTime(&t, c->ev_pool[r.ev], c->ev_pool[r.ev + 1]) != cudaSuccess) { cudaGetLastError(); continue; }
        ms[r.kind] += t; cnt[r.kind] += 1;
    }
    double fl_useful = 0, fl_padded = 0, gbytes_w = 0, sbytes = 0, natoms = 0;
    const size_t es = elem_size(c), vs = c->val_dtype == NOLSM_DTYPE_F64 ? 8 : 4;
    for (auto& pr : c->prof_ranges) {
        const int64_t cntA = pr.second - pr.first;
        std::vector<int32_t> gm(cntA);
        CU_TRY(c, cudaMemcpy(gm.data(), c->a_gemms + pr.first, 4 * cntA, cudaMemcpyDeviceToHost));
        for (int64_t a = pr.first; a < pr.second; ++a) {
            MatInfo mi;
            fill_matinfo(c, a, mi);
            const double d = mi.n;
            fl_useful += 2.0 * d * d * d * gm[a - pr.first];
            const double pm = (double)((mi.n + BM - 1) / BM) * BM, pn = (double)mi.ntn * mi.bn, pk = (double)((mi.n + 15) / 16) * 16;
            fl_padded += 2.0 * pm * pn * pk * gm[a - pr.first];
            gbytes_w += 2.0 * d * mi.ld * es;
            const double nv = (double)(c->blk_off[c->row_ptr[a + 1]] - c->blk_off[c->row_ptr[a]]);
            sbytes += nv * (c->last_ds + vs) + d * mi.ld * es + d * mi.nbi * es;
            natoms += 1;
        }
    }
    unsigned long long ge = 0;
    CU_TRY(c, cudaMemcpy(&ge, c->d_gather_elems, 8, cudaMemcpyDeviceToHost));
    out[0] = ms[K_GATHER]; out[1] = cnt[K_GATHER]; out[2] = gbytes_w + (double)ge * vs;
    out[3] = ms[K_GEMM]; out[4] = cnt[K_GEMM]; out[5] = fl_useful; out[6] = fl_padded;
    out[7] = ms[K_DCOLS]; out[8] = cnt[K_DCOLS]; out[9] = sbytes;
    out[10] = ms[K_OTHER]; out[11] = cnt[K_OTHER];
    out[12] = natoms; out[13] = (double)c->launches;
    return NOLSM_OK;
}

}  // extern "C"
