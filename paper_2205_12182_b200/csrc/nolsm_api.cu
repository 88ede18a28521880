// C ABI of the NOLSM hot path (include/nolsm.h): context, assemble (a0), batch orchestration of the
// device pipeline (a1-a7) and diagnostics. Host code only plans and launches; every step of the path
// runs in the kernels of kernels.cuh and gemm_umma.cuh.
#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <thread>
#include <vector>

#include "../../include/nolsm.h"
#include "gemm2sm.cuh"
#include "kernels.cuh"
#include "persist.cuh"
#include "tmap_host.h"

using namespace nolsm;

namespace {

template <typename F>
void parallel_for(int64_t n, F f) {
    unsigned nt = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
    if (n < 1 << 11) nt = 1;
    if (nt == 1) { f(0, n); return; }
    std::vector<std::thread> th;
    const int64_t chunk = (n + nt - 1) / nt;
    for (unsigned t = 0; t < nt; ++t) {
        const int64_t b = t * chunk, e = std::min<int64_t>(n, b + chunk);
        if (b < e) th.emplace_back([=] { f(b, e); });
    }
    for (auto& x : th) x.join();
}

enum { K_GATHER = 0, K_GEMM = 1, K_DCOLS = 2, K_OTHER = 3 };
constexpr int ROUND_DEPTH = 4;    // rounds kept in flight ahead of the device

}  // namespace

struct nolsm_ctx {
    int dev = 0;
    nolsm_options opt{};
    std::string err;
    bool assembled = false;
    int sms = 148;

    // host copy of the pattern and derived index data
    int64_t n_atoms = 0, nnzb = 0, nvals = 0;
    std::vector<int32_t> atom_nb, col_idx, nset_atom, nset_slot, nset_off, dim, pos;
    std::vector<int64_t> row_ptr, blk_off, nset_ptr;
    bool filtered = false;
    // units (C-19): unit u serves the atoms unit_mem[unit_ptr[u] .. unit_ptr[u+1]) with one submatrix on uset
    int64_t n_units = 0;
    std::vector<int64_t> unit_ptr, uset_ptr;
    std::vector<int32_t> unit_mem, uset_atom, uset_off, udim, upos, unit_of, nset_uoff;
    long long *d_unit_ptr = nullptr, *d_uset_ptr = nullptr;
    int *d_unit_mem = nullptr, *d_uset_atom = nullptr, *d_uset_off = nullptr, *d_udim = nullptr, *d_upos = nullptr, *d_nset_uoff = nullptr;
    bool combined = false;
    int* d_feed = nullptr;              // units of the running call (combined mode)
    std::vector<int32_t> h_feed;
    int max_n = 0, max_nset = 0, max_nbi = 0;

    // device arrays
    std::vector<std::pair<void*, size_t>> owned;   // everything cudaMalloc'ed by assemble
    std::vector<std::pair<void*, size_t>> pool;    // blocks of the previous assemble, reused by the next one (cudaFree of GB-sized
                                                   // blocks stalled re-assembly for up to 0.7 s; freed by nolsm_destroy)
    long long *d_row_ptr = nullptr, *d_blk_off = nullptr, *d_nset_ptr = nullptr;
    int *d_col_idx = nullptr, *d_atom_nb = nullptr, *d_nset_atom = nullptr, *d_nset_slot = nullptr, *d_nset_off = nullptr;
    const void *dH = nullptr, *dS = nullptr;
    int val_dtype = NOLSM_DTYPE_F64;

    // engine (nolsm_device.cuh): slots, op tables, feed, workspace, tensor maps
    Engine eng{};
    void* ws = nullptr;
    size_t ws_bytes = 0;
    CUtensorMap* d_maps = nullptr;
    float *d_vec = nullptr, *d_nrm = nullptr;
    int* h_done = nullptr;              // pinned, mapped
    int *d_dim = nullptr, *d_pos = nullptr;
    double* d_e_atom = nullptr;
    double* d_q_atom = nullptr;
    cudaStream_t s_main = nullptr, s_x = nullptr, s_f = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_x = nullptr, ev_f = nullptr, ev_in = nullptr, ev_out = nullptr;
    cudaEvent_t ev_round[ROUND_DEPTH] = {};
    cudaGraphExec_t graph_exec = nullptr;
    bool use_graph = true;

    // persistent engine (persist.cuh): one kernel launch per density_matrix call
    bool persist = false;
    PEngine peng{};
    int* d_abort = nullptr;
    signed char* d_die = nullptr;       // [256] SM -> L2 die table of the die probe (persistent engine)
    int ndie = 1;
    int p_grid = 0;                     // CTAs of the persistent kernel: 4 x the clusters that can be resident together
    cudaEvent_t ev_k0 = nullptr, ev_k1 = nullptr;
    int h_a0 = 0;
    unsigned long long h_ctr0[PC_LEN] = {};
    std::vector<unsigned int> h_sclaim0;
    bool last_persist = false;
    double timeout_s = 300.0;

    // last density call
    cudaStream_t last_stream = nullptr;
    int64_t last_a0 = 0, last_a1 = 0;
    bool have_result = false;
    void* d_D_stage = nullptr;
    size_t d_D_stage_bytes = 0;
    size_t last_ds = 8;
    int64_t rounds = 0;

    // sampled per-launch profiling (options.profile_every): CUDA events on the launching stream
    struct Rec { int kind; size_t ev; };
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    std::vector<Rec> recs;
    bool prof_on = false;
    int64_t launches = 0;
};

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
bool sync_debug() {                                   // NOLSM_SYNC_DEBUG: eager rounds (NOLSM_GRAPH=0) name and synchronise every launch
    static const bool on = getenv("NOLSM_SYNC_DEBUG") != nullptr;
    return on;
}
void prof_end(nolsm_ctx* c, size_t i, cudaStream_t s) {
    if (c->prof_on) cudaEventRecord(c->ev_pool[i + 1], s);
    if (sync_debug()) {
        const cudaError_t e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) { fprintf(stderr, "nolsm: launch %lld failed: %s\n", (long long)c->launches, cudaGetErrorString(e)); abort(); }
    }
}

#define LAUNCH(c, kind, s, ...)                      \
    do {                                             \
        const size_t pi_ = prof_begin(c, kind, s);   \
        if (sync_debug()) fprintf(stderr, "nolsm: launch %lld kind %d: %s\n", (long long)(c)->launches, kind, #__VA_ARGS__); \
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
    bytes = std::max<size_t>(bytes, 16);
    // best fit from the pool: the smallest block that holds `bytes` and is not more than twice as large
    int best = -1;
    for (int i = 0; i < (int)c->pool.size(); ++i)
        if (c->pool[i].second >= bytes && c->pool[i].second <= 2 * bytes + 4096 && (best < 0 || c->pool[i].second < c->pool[best].second)) best = i;
    if (best >= 0) {
        *p = c->pool[best].first;
        c->owned.push_back(c->pool[best]);
        c->pool.erase(c->pool.begin() + best);
        return NOLSM_OK;
    }
    cudaError_t e = cudaMalloc(p, bytes);
    if (e == cudaErrorMemoryAllocation && !c->pool.empty()) {      // give the pooled blocks back and try once more
        cudaGetLastError();
        for (auto& b : c->pool) cudaFree(b.first);
        c->pool.clear();
        e = cudaMalloc(p, bytes);
    }
    CU_TRY(c, e);
    c->owned.push_back({*p, bytes});
    return NOLSM_OK;
}

// Ends the assembled state. The device blocks go to the pool (release = true: back to the driver).
void free_assembled(nolsm_ctx* c, bool release = false) {
    for (auto& b : c->owned) c->pool.push_back(b);
    c->owned.clear();
    if (release) {
        for (auto& b : c->pool) cudaFree(b.first);
        c->pool.clear();
        if (c->h_done) { cudaFreeHost(c->h_done); c->h_done = nullptr; }
    }
    if (c->d_D_stage && release) { cudaFree(c->d_D_stage); c->d_D_stage = nullptr; c->d_D_stage_bytes = 0; }
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    c->ws = nullptr; c->assembled = false; c->have_result = false;
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

// The persistent engine serves the mixed-precision tcgen05 path; the round engine serves the FP32 / SIMT
// validation modes (and NOLSM_ENGINE=rounds).
bool want_persist(const nolsm_ctx* c) {
    if (!use_umma(c)) return false;
    if (c->opt.engine == NOLSM_ENGINE_ROUNDS) return false;
    return true;
}

SysView sys_view(const nolsm_ctx* c) {
    SysView v;
    v.row_ptr = c->d_row_ptr; v.col_idx = c->d_col_idx; v.blk_off = c->d_blk_off; v.atom_nb = c->d_atom_nb;
    v.nset_ptr = c->d_nset_ptr; v.nset_atom = c->d_nset_atom; v.nset_slot = c->d_nset_slot; v.nset_off = c->d_nset_off;
    v.unit_ptr = c->d_unit_ptr; v.unit_mem = c->d_unit_mem; v.uset_ptr = c->d_uset_ptr; v.uset_atom = c->d_uset_atom;
    v.uset_off = c->d_uset_off; v.nset_uoff = c->d_nset_uoff;
    return v;
}

size_t gather_smem(int max_nset, int cap) { return (size_t)max_nset * 8 + (size_t)(max_nset + 1) * 4 + (size_t)cap * 2 + 16; }

template <typename T>
int launch_gather(nolsm_ctx* c, const Engine& e, int max_nset, cudaStream_t s) {
    const size_t smem = gather_smem(max_nset, e.cap);
    dim3 grid(std::min(max_nset, 48), e.S, 2);
    if (c->val_dtype == NOLSM_DTYPE_F64) {
        auto k = k_gather<double, T>;
        LAUNCH(c, K_GATHER, s, k<<<grid, 256, smem, s>>>(e, sys_view(c), (const double*)c->dS, (const double*)c->dH, (T*)c->ws, max_nset));
    } else {
        auto k = k_gather<float, T>;
        LAUNCH(c, K_GATHER, s, k<<<grid, 256, smem, s>>>(e, sys_view(c), (const float*)c->dS, (const float*)c->dH, (T*)c->ws, max_nset));
    }
    return NOLSM_OK;
}

template <typename T>
void launch_gemm(nolsm_ctx* c, const Engine& e, int launch, cudaStream_t s) {
    if (use_umma(c)) {
        UmmaArgs a;
        a.e = e; a.maps = c->d_maps; a.base = (__half*)c->ws; a.launch = launch;
        LAUNCH(c, K_GEMM, s, gemm2_round_kernel<<<c->sms & ~1, G2_CTRL_THREADS, G2_SMEM_BYTES, s>>>(a));
    } else {
        const int t64 = (e.cap + 63) / 64;
        LAUNCH(c, K_GEMM, s, k_gemm_simt<T><<<dim3(t64 * t64, e.S), 256, 0, s>>>(e, (T*)c->ws, launch));
    }
}

size_t dcols_smem(const nolsm_ctx* c) { return (size_t)(c->max_nset + 1) * 4 + (size_t)c->max_n * c->max_nbi * 4 + 16; }

template <typename T, typename TD>
void launch_dcols(nolsm_ctx* c, const Engine& e, TD* D, cudaStream_t s) {
    const size_t smem = dcols_smem(c);
    const int gx = std::max(1, std::min((c->max_n + 7) / 8, 12));
    dim3 grid(gx, e.S);
    if (c->val_dtype == NOLSM_DTYPE_F64) {
        auto k = k_dcols_scatter<T, double, TD>;
        LAUNCH(c, K_DCOLS, s, k<<<grid, 256, smem, s>>>(e, sys_view(c), (const T*)c->ws, (const double*)c->dH, (const double*)c->dS, D, c->d_e_atom, c->d_q_atom, c->max_nset));
    } else {
        auto k = k_dcols_scatter<T, float, TD>;
        LAUNCH(c, K_DCOLS, s, k<<<grid, 256, smem, s>>>(e, sys_view(c), (const T*)c->ws, (const float*)c->dH, (const float*)c->dS, D, c->d_e_atom, c->d_q_atom, c->max_nset));
    }
}

// Raises the dynamic shared memory limits of the templated kernels once per assemble (must not happen
// during stream capture).
template <typename T>
int set_smem_limits(nolsm_ctx* c) {
    const int g = (int)std::max<size_t>(gather_smem(c->max_nset, c->eng.cap), 48 * 1024);
    const int d = (int)std::max<size_t>(dcols_smem(c), 48 * 1024);
    if (d > 227 * 1024) return fail(c, NOLSM_EINVAL, "n_i * nb(i) too large for the D-columns kernel");
    CU_TRY(c, cudaFuncSetAttribute(k_gather<double, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, g));
    CU_TRY(c, cudaFuncSetAttribute(k_gather<float, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, g));
    CU_TRY(c, cudaFuncSetAttribute(k_dcols_scatter<T, double, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, d));
    CU_TRY(c, cudaFuncSetAttribute(k_dcols_scatter<T, double, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, d));
    CU_TRY(c, cudaFuncSetAttribute(k_dcols_scatter<T, float, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, d));
    CU_TRY(c, cudaFuncSetAttribute(k_dcols_scatter<T, float, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, d));
    return NOLSM_OK;
}

// One round (nolsm_device.cuh). forked == true: three concurrent branches (used under stream capture):
//   s_main: round begin -> GEMM launch 0 -> GEMM launch 1 ;  s_x: gather + power iterations + first Schulz step ;
//   s_f: D columns + scatter.  forked == false: the same kernels serially on s_main (profiled rounds).
template <typename T>
int enqueue_round(nolsm_ctx* c, const Engine& e, void* D, int d_dtype, bool forked) {
    cudaStream_t sm = c->s_main, sx = forked ? c->s_x : c->s_main, sf = forked ? c->s_f : c->s_main;
    LAUNCH(c, K_OTHER, sm, k_round_begin<<<1, MAX_SLOTS, 0, sm>>>(e));
    if (forked) {
        CU_TRY(c, cudaEventRecord(c->ev_fork, sm));
        CU_TRY(c, cudaStreamWaitEvent(sx, c->ev_fork, 0));
        CU_TRY(c, cudaStreamWaitEvent(sf, c->ev_fork, 0));
    }
    // branch s_f: a6 + a7 for the slots in phase FIN
    if (d_dtype == NOLSM_DTYPE_F64) launch_dcols<T, double>(c, e, (double*)D, sf);
    else launch_dcols<T, float>(c, e, (float*)D, sf);
    // branch s_x: a1 for the slots in phase NEW, power iterations for NEW (S) and PA (A)
    int r;
    if ((r = launch_gather<T>(c, e, c->max_nset, sx))) return r;
    const int P = std::max(e.p_s, e.p_a);
    LAUNCH(c, K_OTHER, sx, k_vec_init<<<dim3((e.cap + 255) / 256, e.S), 256, 0, sx>>>(e, c->d_vec, c->d_nrm, P));
    for (int it = 0; it < P; ++it)
        LAUNCH(c, K_OTHER, sx, k_matvec<T><<<dim3(16, e.S), 256, 0, sx>>>(e, (const T*)c->ws, c->d_vec, c->d_nrm, it));
    LAUNCH(c, K_OTHER, sx, k_power_finish<T><<<dim3(32, e.S), 256, 0, sx>>>(e, (T*)c->ws, c->d_nrm));
    // main branch: the two grouped GEMM launches of the round
    launch_gemm<T>(c, e, 0, sm);
    launch_gemm<T>(c, e, 1, sm);
    if (forked) {
        CU_TRY(c, cudaEventRecord(c->ev_x, sx));
        CU_TRY(c, cudaEventRecord(c->ev_f, sf));
        CU_TRY(c, cudaStreamWaitEvent(sm, c->ev_x, 0));
        CU_TRY(c, cudaStreamWaitEvent(sm, c->ev_f, 0));
    }
    CU_TRY(c, cudaGetLastError());
    return NOLSM_OK;
}

// Waits for the last density_matrix call. The persistent kernel is watched: past the time limit the host
// raises the kernel's abort word (copy on a second stream), which makes every role leave its loop.
int wait_result(nolsm_ctx* c) {
    if (c->last_persist) {
        const auto t0 = std::chrono::steady_clock::now();
        bool aborted = false;
        for (;;) {
            const cudaError_t q = cudaEventQuery(c->ev_out);
            if (q == cudaSuccess) break;
            if (q != cudaErrorNotReady) { c->err = std::string("persistent engine: ") + cudaGetErrorString(q); return NOLSM_ECUDA; }
            const double el = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
            if (!aborted && el > c->timeout_s) {
                static const int one = 1;
                cudaMemcpyAsync(c->d_abort, &one, 4, cudaMemcpyHostToDevice, c->s_x);
                aborted = true;
            }
            if (el > c->timeout_s + 20.0) { c->err = "persistent engine did not stop after abort"; return NOLSM_ECUDA; }
            std::this_thread::sleep_for(std::chrono::microseconds(el < 0.01 ? 20 : 200));
        }
        if (aborted) { c->err = "persistent engine exceeded its time limit and was aborted"; return NOLSM_ECUDA; }
    }
    CU_TRY(c, cudaStreamSynchronize(c->last_stream));
    return NOLSM_OK;
}

int getenv_int(const char* name, int dflt);

// ---- submatrix combination (Eq. 9 / Eq. 10; C-19). Integer arithmetic only. ----
int64_t combine_cost(int64_t n, int mode) {
    if (mode == 1) return n * n * n;                               // Eq. 9: FLOP of a dense multiplication
    const int64_t n16 = (n + 15) / 16 * 16, t = (n16 + 255) / 256;  // Eq. 10 with the engine's tile-time characteristic
    return t * t * ((n16 + 63) / 64);
}
// sum of nb over the atoms two ascending lists have in common
int64_t overlap_dim(const int32_t* a, int64_t na, const int32_t* b, int64_t nb_, const int32_t* atom_nb) {
    int64_t i = 0, j = 0, d = 0;
    while (i < na && j < nb_) {
        if (a[i] < b[j]) ++i;
        else if (a[i] > b[j]) ++j;
        else { d += atom_nb[a[i]]; ++i; ++j; }
    }
    return d;
}
// Builds the units of the context from the per-atom index sets: greedy groups (mode 1 / 2) or one atom per unit (mode 0).
void build_units(nolsm_ctx* c, int mode, int max_dim, int max_members, int max_cand) {
    const int64_t n_at = c->n_atoms;
    const int32_t* nb = c->atom_nb.data();
    c->unit_ptr.assign(1, 0); c->unit_mem.clear(); c->uset_ptr.assign(1, 0); c->uset_atom.clear(); c->uset_off.clear(); c->udim.clear();
    c->unit_of.assign(n_at, -1); c->upos.assign(n_at, 0);
    const bool verbose = getenv_int("NOLSM_VERBOSE", 0) >= 2;
    auto t_prev = std::chrono::steady_clock::now();
    auto lap = [&](const char* what) {
        if (!verbose) return;
        const auto t = std::chrono::steady_clock::now();
        fprintf(stderr, "  build_units: %-24s %8.2f ms\n", what, std::chrono::duration<double, std::milli>(t - t_prev).count());
        t_prev = t;
    };
    std::vector<char> is_free(n_at, 1);
    std::vector<int32_t> G, gw(n_at, 0);      // gw[k] = n_b(k) while atom k is in the current group's set, else 0
    std::vector<std::pair<int64_t, int32_t>> cand;
    // overlaps dim(N(i) & N(j)) of every pair of the pattern, in parallel (the greedy pass below is sequential)
    std::vector<int32_t> ov;
    if (mode != 0 && max_members > 1) {
        ov.resize(c->nset_atom.size());
        // the overlap is symmetric: each thread computes the pairs j > i of its atoms and stores both directions (the
        // position of i in the sorted N(j) by binary search). w[k] = n_b(k) while k is in N(i), else 0: one gather per term.
        parallel_for(n_at, [&](int64_t b, int64_t e) {
            std::vector<int32_t> w(n_at, 0);
            for (int64_t i = b; i < e; ++i) {
                const int32_t* Ni = c->nset_atom.data() + c->nset_ptr[i];
                const int64_t ni = c->nset_ptr[i + 1] - c->nset_ptr[i];
                for (int64_t q = 0; q < ni; ++q) w[Ni[q]] = nb[Ni[q]];
                for (int64_t q = 0; q < ni; ++q) {
                    const int32_t j = Ni[q];
                    if (j <= i) { if (j == i) ov[c->nset_ptr[i] + q] = 0; continue; }
                    const int32_t* Nj = c->nset_atom.data() + c->nset_ptr[j];
                    const int64_t nj = c->nset_ptr[j + 1] - c->nset_ptr[j];
                    int32_t d = 0;
                    for (int64_t t = 0; t < nj; ++t) d += w[Nj[t]];
                    ov[c->nset_ptr[i] + q] = d;
                    const int32_t* it = std::lower_bound(Nj, Nj + nj, (int32_t)i);     // the pattern is symmetric (validated in assemble)
                    if (it != Nj + nj && *it == (int32_t)i) ov[c->nset_ptr[j] + (it - Nj)] = d;
                }
                for (int64_t q = 0; q < ni; ++q) w[Ni[q]] = 0;
            }
        });
    }
    lap("pair overlaps");
    for (int64_t i = 0; i < n_at; ++i) {
        if (!is_free[i]) continue;
        is_free[i] = 0;
        const int32_t* Ni = c->nset_atom.data() + c->nset_ptr[i];
        const int64_t ni = c->nset_ptr[i + 1] - c->nset_ptr[i];
        const size_t m0 = c->unit_mem.size();
        c->unit_mem.push_back((int32_t)i);
        G.assign(Ni, Ni + ni);
        int64_t n_g = c->dim[i];
        if (mode != 0 && max_members > 1) {
            for (int64_t q = 0; q < ni; ++q) gw[Ni[q]] = nb[Ni[q]];
            cand.clear();
            for (int64_t q = 0; q < ni; ++q) {
                const int32_t j = Ni[q];
                if (j == i || !is_free[j]) continue;
                cand.emplace_back(-(int64_t)ov[c->nset_ptr[i] + q], j);
            }
            std::sort(cand.begin(), cand.end());
            if ((int)cand.size() > max_cand) cand.resize(max_cand);
            for (const auto& cj : cand) {
                if ((int)(c->unit_mem.size() - m0) >= max_members) break;
                const int32_t j = cj.second;
                const int32_t* Nj = c->nset_atom.data() + c->nset_ptr[j];
                const int64_t nj = c->nset_ptr[j + 1] - c->nset_ptr[j];
                int64_t n_gj = -cj.first;                   // while the set is still N(i): the pair overlap computed above
                if (G.size() != (size_t)ni) { n_gj = 0; for (int64_t t = 0; t < nj; ++t) n_gj += gw[Nj[t]]; }
                const int64_t n_u = n_g + c->dim[j] - n_gj;
                if (n_u > max_dim) continue;
                if (combine_cost(n_u, mode) < combine_cost(n_g, mode) + combine_cost(c->dim[j], mode)) {
                    c->unit_mem.push_back(j);
                    is_free[j] = 0;
                    for (int64_t t = 0; t < nj; ++t)
                        if (gw[Nj[t]] == 0) { gw[Nj[t]] = nb[Nj[t]]; G.push_back(Nj[t]); }
                    n_g = n_u;
                }
            }
            for (int32_t a : G) gw[a] = 0;
            if (c->unit_mem.size() - m0 > 1) std::sort(G.begin(), G.end());
        }
        const int32_t u = (int32_t)c->udim.size();
        int off = 0;
        for (int32_t a : G) { c->uset_atom.push_back(a); c->uset_off.push_back(off); off += nb[a]; }
        c->uset_ptr.push_back((int64_t)c->uset_atom.size());
        c->unit_ptr.push_back((int64_t)c->unit_mem.size());
        c->udim.push_back(off);
        for (size_t m = m0; m < c->unit_mem.size(); ++m) c->unit_of[c->unit_mem[m]] = u;
    }
    c->n_units = (int64_t)c->udim.size();
    lap("greedy pass");
    // offsets of every atom of N(i) inside the matrix of i's unit (N(i) is a subset of the unit's set: one merge walk)
    c->nset_uoff.resize(c->nset_atom.size());
    for (int64_t i = 0; i < n_at; ++i) {
        const int32_t u = c->unit_of[i];
        int64_t g = c->uset_ptr[u];
        for (int64_t q = c->nset_ptr[i]; q < c->nset_ptr[i + 1]; ++q) {
            while (c->uset_atom[g] != c->nset_atom[q]) ++g;
            c->nset_uoff[q] = c->uset_off[g];
            if (c->nset_atom[q] == i) c->upos[i] = c->uset_off[g];
        }
    }
}

// Runs k_die_probe and builds the SM -> die table (persist.cuh). Leaves ndie = 1 (no affinity) when the
// near / far pattern is not a clean two-way split of the SMs.
void probe_dies(nolsm_ctx* c) {
    c->ndie = 1;
    if (getenv_int("NOLSM_DIE_AFFINITY", 0) == 0) return;   // off by default: measured on B200, affinity does not change the DRAM traffic
    unsigned long long* d_lines = nullptr;
    unsigned int* d_best = nullptr;
    std::vector<unsigned int> best(256 * NPROBE, 0xFFFFFFFFu);
    if (cudaMalloc((void**)&d_lines, NPROBE * 2048) != cudaSuccess || cudaMalloc((void**)&d_best, best.size() * 4) != cudaSuccess ||
        cudaMalloc((void**)&c->d_die, 256) != cudaSuccess) { cudaGetLastError(); cudaFree(d_lines); cudaFree(d_best); return; }
    cudaMemset(d_lines, 0, NPROBE * 2048);
    cudaMemcpy(d_best, best.data(), best.size() * 4, cudaMemcpyHostToDevice);
    for (int rep = 0; rep < 4; ++rep) k_die_probe<<<c->sms * 6, 32>>>(d_lines, d_best);
    const bool ok = cudaDeviceSynchronize() == cudaSuccess &&
                    cudaMemcpy(best.data(), d_best, best.size() * 4, cudaMemcpyDeviceToHost) == cudaSuccess;
    cudaFree(d_lines); cudaFree(d_best);
    std::vector<signed char> die(256, (signed char)-1);
    if (ok) {
        std::vector<int> sms;
        for (int sm = 0; sm < 256; ++sm) if (best[sm * NPROBE] != 0xFFFFFFFFu) sms.push_back(sm);
        if (getenv_int("NOLSM_VERBOSE", 0) >= 2)
            for (int sm : sms) {
                fprintf(stderr, "probe sm %3d:", sm);
                for (int l = 0; l < NPROBE; ++l) fprintf(stderr, " %5.1f", best[sm * NPROBE + l] / 64.0);
                fprintf(stderr, "\n");
            }
        // M[sm][line] = latency with the SM's mean and the line's mean removed (an SM's distance to the L2 slices
        // and a line's slice position shift whole rows / columns); what is left is +-(near/far gap)/2 with the sign
        // given by (die of SM) xor (home die of line): a rank-one +-1 pattern. Its leading left singular vector
        // (power iteration on M M^T) splits the SMs by die.
        const int ns = (int)sms.size();
        if (ns == c->sms && ns >= 8) {
            std::vector<double> M((size_t)ns * NPROBE);
            for (int i = 0; i < ns; ++i) for (int l = 0; l < NPROBE; ++l) M[(size_t)i * NPROBE + l] = best[sms[i] * NPROBE + l] / 64.0;
            for (int i = 0; i < ns; ++i) {
                double m = 0; for (int l = 0; l < NPROBE; ++l) m += M[(size_t)i * NPROBE + l];
                m /= NPROBE; for (int l = 0; l < NPROBE; ++l) M[(size_t)i * NPROBE + l] -= m;
            }
            for (int l = 0; l < NPROBE; ++l) {
                double m = 0; for (int i = 0; i < ns; ++i) m += M[(size_t)i * NPROBE + l];
                m /= ns; for (int i = 0; i < ns; ++i) M[(size_t)i * NPROBE + l] -= m;
            }
            std::vector<double> u(ns), v(NPROBE);
            for (int i = 0; i < ns; ++i) u[i] = M[(size_t)i * NPROBE];          // start: the first line's pattern
            double sigma = 0, total = 0;
            for (double x : M) total += x * x;
            for (int it = 0; it < 50; ++it) {
                for (int l = 0; l < NPROBE; ++l) { double a = 0; for (int i = 0; i < ns; ++i) a += M[(size_t)i * NPROBE + l] * u[i]; v[l] = a; }
                double nv = 0; for (double x : v) nv += x * x; nv = std::sqrt(nv) + 1e-300; for (double& x : v) x /= nv;
                for (int i = 0; i < ns; ++i) { double a = 0; for (int l = 0; l < NPROBE; ++l) a += M[(size_t)i * NPROBE + l] * v[l]; u[i] = a; }
                double nu = 0; for (double x : u) nu += x * x; sigma = std::sqrt(nu); for (double& x : u) x /= (sigma + 1e-300);
            }
            std::vector<double> au(ns);
            for (int i = 0; i < ns; ++i) au[i] = std::fabs(u[i]);
            std::nth_element(au.begin(), au.begin() + ns / 2, au.end());
            const double med = au[ns / 2];
            int n1 = 0, weak = 0;
            for (int i = 0; i < ns; ++i) {
                die[sms[i]] = (signed char)(u[i] > 0 ? 1 : 0);
                n1 += u[i] > 0;
                weak += std::fabs(u[i]) < 0.3 * med;
            }
            const double explained = sigma * sigma / (total + 1e-300);
            if (explained > 0.5 && weak <= ns / 20 && n1 * 10 >= ns * 4 && n1 * 10 <= ns * 6) c->ndie = 2;
            if (getenv_int("NOLSM_VERBOSE", 0))
                fprintf(stderr, "nolsm: die probe: %d SMs, %d on die 1, %d weak, rank-one part explains %.0f %% of the variance -> ndie = %d\n",
                        ns, n1, weak, 100.0 * explained, c->ndie);
        } else if (getenv_int("NOLSM_VERBOSE", 0)) fprintf(stderr, "nolsm: die probe: %d SMs seen of %d -> no affinity\n", ns, c->sms);
    }
    if (c->ndie != 2) std::fill(die.begin(), die.end(), (signed char)-1);
    cudaMemcpy(c->d_die, die.data(), 256, cudaMemcpyHostToDevice);
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
    if (o.power_iters_s < 0) o.power_iters_s = 0;      // 0 = default of the engine that runs (assemble)
    if (o.power_iters_a < 0) o.power_iters_a = 0;
    if (o.eps_filter < 0) { delete c; return NOLSM_EINVAL; }
    if (o.sign_scaled_iters == 0) o.sign_scaled_iters = 6;
    if (getenv("NOLSM_SIGN_SCALED_ITERS")) o.sign_scaled_iters = getenv_int("NOLSM_SIGN_SCALED_ITERS", 6);
    if (o.sign_scaled_iters < 0) o.sign_scaled_iters = 0;
    if (o.sign_scaled_iters > 14) o.sign_scaled_iters = 14;
    if (getenv("NOLSM_COMBINE")) o.combine = getenv_int("NOLSM_COMBINE", 0);
    if (o.combine < 0 || o.combine > 2) { delete c; return NOLSM_EINVAL; }
    if (o.combine_max_dim <= 0) o.combine_max_dim = getenv_int("NOLSM_COMBINE_MAX_DIM", 2048);
    if (o.combine_max_members <= 0) o.combine_max_members = getenv_int("NOLSM_COMBINE_MAX_MEMBERS", 16);
    if (o.combine_max_candidates <= 0) o.combine_max_candidates = getenv_int("NOLSM_COMBINE_MAX_CANDIDATES", 24);
    if (getenv_int("NOLSM_CLUSTER", 0) > 0) o.cluster_ctas = getenv_int("NOLSM_CLUSTER", 0);
    if (o.cluster_ctas != 0 && o.cluster_ctas != 2 && o.cluster_ctas != 4) { delete c; return NOLSM_EINVAL; }
    if (o.sign_scale == 0.f) o.sign_scale = 1.5f;
    if (const char* v = getenv("NOLSM_SIGN_SCALE")) o.sign_scale = (float)atof(v);
    if (!(o.sign_scale > 1.f && o.sign_scale < 1.7320508f)) { delete c; return NOLSM_EINVAL; }
    cudaSetDevice(cuda_device);
    cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, cuda_device);
    if (getenv_int("NOLSM_PROFILE_EVERY", 0) > 0) o.profile_every = getenv_int("NOLSM_PROFILE_EVERY", 0);
    if (getenv_int("NOLSM_SLOTS", 0) > 0) o.batch_atoms = getenv_int("NOLSM_SLOTS", 0);
    c->use_graph = getenv_int("NOLSM_GRAPH", 1) != 0;
    if (const char* en = getenv("NOLSM_ENGINE")) {
        if (!strcmp(en, "rounds")) o.engine = NOLSM_ENGINE_ROUNDS;
        else if (!strcmp(en, "persistent")) o.engine = NOLSM_ENGINE_PERSISTENT;
    }
    if (o.engine < 0 || o.engine > NOLSM_ENGINE_ROUNDS) { delete c; return NOLSM_EINVAL; }
    if (getenv_int("NOLSM_TIMEOUT_S", 0) > 0) c->timeout_s = getenv_int("NOLSM_TIMEOUT_S", 0);
    bool ok = cudaStreamCreateWithFlags(&c->s_main, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->s_x, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->s_f, cudaStreamNonBlocking) == cudaSuccess;
    cudaEvent_t* evs[] = {&c->ev_fork, &c->ev_x, &c->ev_f, &c->ev_in, &c->ev_out};
    for (cudaEvent_t* e : evs) ok = ok && cudaEventCreateWithFlags(e, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < ROUND_DEPTH; ++i) ok = ok && cudaEventCreateWithFlags(&c->ev_round[i], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaEventCreate(&c->ev_k0) == cudaSuccess && cudaEventCreate(&c->ev_k1) == cudaSuccess;
    if (!ok) { cudaGetLastError(); delete c; return NOLSM_ECUDA; }
    if (use_umma(c)) {
        if (cudaFuncSetAttribute(gemm2_round_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, G2_SMEM_BYTES) != cudaSuccess ||
            cudaFuncSetAttribute(nolsm_persist_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SMEM_BYTES) != cudaSuccess ||
            cudaFuncSetAttribute(nolsm_persist_kernel<G4_CTAS>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SMEM_BYTES) != cudaSuccess) {
            cudaGetLastError();
            delete c;
            return NOLSM_ECUDA;
        }
    }
    if (use_umma(c) && o.engine != NOLSM_ENGINE_ROUNDS) probe_dies(c);
    *out = c;
    return NOLSM_OK;
}

int nolsm_destroy(nolsm_ctx* c) {
    if (!c) return NOLSM_EINVAL;
    cudaSetDevice(c->dev);
    free_assembled(c, true);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    cudaEvent_t evs[] = {c->ev_fork, c->ev_x, c->ev_f, c->ev_in, c->ev_out, c->ev_k0, c->ev_k1};
    for (cudaEvent_t e : evs) if (e) cudaEventDestroy(e);
    for (int i = 0; i < ROUND_DEPTH; ++i) if (c->ev_round[i]) cudaEventDestroy(c->ev_round[i]);
    if (c->d_die) cudaFree(c->d_die);
    if (c->s_main) cudaStreamDestroy(c->s_main);
    if (c->s_x) cudaStreamDestroy(c->s_x);
    if (c->s_f) cudaStreamDestroy(c->s_f);
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
    const bool verbose = getenv_int("NOLSM_VERBOSE", 0) >= 1;
    auto t_prev = std::chrono::steady_clock::now();
    auto lap = [&](const char* what) {
        if (!verbose) return;
        const auto t = std::chrono::steady_clock::now();
        fprintf(stderr, "nolsm_assemble: %-28s %8.2f ms\n", what, std::chrono::duration<double, std::milli>(t - t_prev).count());
        t_prev = t;
    };
    if (c->have_result) wait_result(c);          // the pooled blocks of the last call are about to be reused
    free_assembled(c);
    lap("free");
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

    lap("pattern to host + validate");
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

    lap("block offsets + uploads");
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
    lap("index sets");
    // ---- units: one submatrix per atom, or per group of atoms (Eq. 9 / Eq. 10; C-19) ----
    c->combined = c->opt.combine != 0 && want_persist(c);
    if (c->opt.combine != 0 && !c->combined) return fail(c, NOLSM_EINVAL, "combine needs the persistent engine (FP16/tcgen05 mode)");
    build_units(c, c->combined ? c->opt.combine : 0, std::min(c->opt.combine_max_dim, P_MAX_CAP), c->opt.combine_max_members,
                c->opt.combine_max_candidates);
    lap("units (grouping)");
    int max_n = 0, min_n = 1 << 30, max_nset = 0, max_nbi = 0;
    double mean_tiles = 0, mean_n2 = 0;
    for (int64_t i = 0; i < n_atoms; ++i) max_nbi = std::max(max_nbi, c->atom_nb[i]);
    for (int64_t u = 0; u < c->n_units; ++u) {
        max_n = std::max(max_n, c->udim[u]);
        min_n = std::min(min_n, c->udim[u]);
        max_nset = std::max<int>(max_nset, (int)(c->uset_ptr[u + 1] - c->uset_ptr[u]));
        int ntm, ntn;
        choose_tiling((c->udim[u] + 15) & ~15, ntm, ntn);
        mean_tiles += (double)ntm * ntn;
        mean_n2 += (double)c->udim[u] * c->udim[u];
    }
    mean_tiles /= (double)c->n_units;
    mean_n2 /= (double)c->n_units;
    if (max_n > 65535) return fail(c, NOLSM_EINVAL, "submatrix dimension > 65535 not supported");
    c->max_n = max_n; c->max_nset = max_nset; c->max_nbi = max_nbi;
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
    if ((r = to_device(c, c->dim.data(), sizeof(int32_t) * n_atoms, &tmp, s))) return r;
    c->d_dim = (int*)tmp;
    if ((r = to_device(c, c->pos.data(), sizeof(int32_t) * n_atoms, &tmp, s))) return r;
    c->d_pos = (int*)tmp;
    if ((r = to_device(c, c->unit_ptr.data(), sizeof(int64_t) * (c->n_units + 1), &tmp, s))) return r;
    c->d_unit_ptr = (long long*)tmp;
    if ((r = to_device(c, c->unit_mem.data(), sizeof(int32_t) * n_atoms, &tmp, s))) return r;
    c->d_unit_mem = (int*)tmp;
    if (c->combined) {
        if ((r = to_device(c, c->uset_ptr.data(), sizeof(int64_t) * (c->n_units + 1), &tmp, s))) return r;
        c->d_uset_ptr = (long long*)tmp;
        if ((r = to_device(c, c->uset_atom.data(), sizeof(int32_t) * c->uset_atom.size(), &tmp, s))) return r;
        c->d_uset_atom = (int*)tmp;
        if ((r = to_device(c, c->uset_off.data(), sizeof(int32_t) * c->uset_off.size(), &tmp, s))) return r;
        c->d_uset_off = (int*)tmp;
        if ((r = to_device(c, c->nset_uoff.data(), sizeof(int32_t) * nn, &tmp, s))) return r;
        c->d_nset_uoff = (int*)tmp;
        if ((r = to_device(c, c->udim.data(), sizeof(int32_t) * c->n_units, &tmp, s))) return r;
        c->d_udim = (int*)tmp;
        if ((r = to_device(c, c->upos.data(), sizeof(int32_t) * n_atoms, &tmp, s))) return r;
        c->d_upos = (int*)tmp;
        if ((r = dmalloc(c, (void**)&c->d_feed, 4 * (size_t)c->n_units))) return r;
    } else {                      // unit u is atom u: the unit arrays are the per-atom ones
        c->d_uset_ptr = c->d_nset_ptr; c->d_uset_atom = c->d_nset_atom; c->d_uset_off = c->d_nset_off;
        c->d_nset_uoff = c->d_nset_off; c->d_udim = c->d_dim; c->d_upos = c->d_pos;
    }

    lap("uploads of index data");
    // ---- engine: slots, workspace, tensor maps ----
    Engine& e = c->eng;
    e = Engine{};
    const size_t es = elem_size(c);
    e.cap = (max_n + 15) & ~15;
    e.ld = ((e.cap + 63) & ~63) + 64 * getenv_int("NOLSM_LD_PAD", 0);        // rows start on 128-byte lines: TMA boxes map to whole L2 lines
    e.bufsz = (long long)e.cap * e.ld;
    e.slotsz = e.bufsz * NBUF;
    size_t free_b = 0, total_b = 0;
    CU_TRY(c, cudaMemGetInfo(&free_b, &total_b));
    const size_t slot_bytes = (size_t)e.slotsz * es;
    const size_t cap_bytes = c->opt.workspace_bytes ? c->opt.workspace_bytes : std::min<size_t>(free_b / 2, (size_t)48 << 30);
    // persistent engine: slot buffers must fit the side tasks' shared memory (power-iteration vectors, Y columns)
    const int g_rowatoms = std::max(1, getenv_int("NOLSM_GATHER_ROWATOMS", 4));
    // (gather task: index tables + dense strip; a strip holds at least one dense row)
    c->persist = want_persist(c) && e.cap <= P_MAX_CAP && max_nbi <= NVC &&
                 (size_t)(3 * max_nset + 2) * 4 + (size_t)max_nset * 8 + 32 + G_STRIP_BYTES <= (size_t)P_SIDE_SMEM &&
                 (size_t)e.cap * 2 <= (size_t)G_STRIP_BYTES;
    if (c->combined && !c->persist) return fail(c, NOLSM_EINVAL, "combine: the groups do not fit the persistent engine (dimension or index-set size)");
    if (!c->persist && c->opt.engine == NOLSM_ENGINE_PERSISTENT)
        return fail(c, NOLSM_EINVAL, "the persistent engine needs FP16/tcgen05 mode, submatrix dimensions <= 4096 and at most 16 basis functions per atom");
    // round engine: enough slots for ~16 waves of tiles per GEMM launch; persistent engine: the slots in
    // flight (GEMM chain + side phases), few enough to keep the active iterates in L2
    // heavy-phase cap of the persistent engine: the live iterates of a slot in the GEMM chain are ~3.5 n^2 FP16
    // (X, T, next X / S, Y, R, next Y); the slots inside the chain together may fill L2 (measured on cfg2:
    // 10-14 slots give the same throughput, fewer starve the pairs, more overflow L2 and draw HBM power)
    int l2_bytes = 0;
    cudaDeviceGetAttribute(&l2_bytes, cudaDevAttrL2CacheSize, c->dev);
    if (l2_bytes <= 0) l2_bytes = 64 << 20;
    int g_max = (int)std::floor(1.0 * (double)l2_bytes / (3.5 * mean_n2 * 2.0));
    g_max = std::max(3, std::min(g_max, 48));
    if (getenv_int("NOLSM_GMAX", 0) > 0) g_max = getenv_int("NOLSM_GMAX", 0);
    int S = c->opt.batch_atoms > 0 ? c->opt.batch_atoms
            : c->persist ? std::min(96, g_max + std::max(12, g_max))
                         : (int)std::ceil(16.0 * c->sms / std::max(1.0, mean_tiles));
    S = std::max(S, 2);
    S = (int)std::min<size_t>(S, std::max<size_t>(2, cap_bytes / slot_bytes));
    S = std::min(S, MAX_SLOTS);
    S = (int)std::min<int64_t>(S, std::max<int64_t>(2, c->n_units));
    e.S = S;
    // after the S slots: two vector blocks per slot and one shared start block (block power iteration), cap x VLD each
    const size_t vec_bytes = (size_t)e.cap * VLD * es;
    c->ws_bytes = slot_bytes * S + vec_bytes * (2 * (size_t)S + 1);
    if ((r = dmalloc(c, &c->ws, c->ws_bytes))) return r;
    CU_TRY(c, cudaMemsetAsync(c->ws, 0, c->ws_bytes, s));
    if ((r = dmalloc(c, (void**)&e.slots, sizeof(Slot) * S))) return r;
    if ((r = dmalloc(c, (void**)&e.ops, sizeof(SlotOp) * 2 * S))) return r;
    if ((r = dmalloc(c, (void**)&e.ntiles, 16))) return r;
    if ((r = dmalloc(c, (void**)&e.next_atom, 16))) return r;
    if ((r = dmalloc(c, (void**)&e.finished, 16))) return r;
    if ((r = dmalloc(c, (void**)&e.prof, sizeof(double) * PF_LEN))) return r;
    CU_TRY(c, cudaMemsetAsync(e.slots, 0, sizeof(Slot) * S, s));
    CU_TRY(c, cudaMemsetAsync(e.ops, 0, sizeof(SlotOp) * 2 * S, s));
    CU_TRY(c, cudaMemsetAsync(e.ntiles, 0, 16, s));
    if (!c->h_done) CU_TRY(c, cudaHostAlloc((void**)&c->h_done, 64, cudaHostAllocMapped));
    *c->h_done = 0;
    int* h_done_dev = nullptr;
    CU_TRY(c, cudaHostGetDevicePointer((void**)&h_done_dev, c->h_done, 0));
    e.h_done = h_done_dev;
    e.tol_inv = c->opt.tol_inv; e.tol_sign = c->opt.tol_sign;
    e.max_inv = c->opt.max_inv_iters; e.max_sign = c->opt.max_sign_iters;
    e.p_s = c->opt.power_iters_s > 0 ? c->opt.power_iters_s : 6;
    e.p_a = c->opt.power_iters_a > 0 ? c->opt.power_iters_a : 12;
    const int P = std::max(e.p_s, e.p_a);
    if (P + 1 > 256) return fail(c, NOLSM_EINVAL, "too many power iterations");
    if ((r = dmalloc(c, (void**)&c->d_vec, sizeof(float) * 2 * (size_t)S * e.ld))) return r;
    if ((r = dmalloc(c, (void**)&c->d_nrm, sizeof(float) * (size_t)(P + 1) * S))) return r;
    int** res_i[] = {&e.at.inv, &e.at.sign, &e.at.status, &e.at.gemms};
    for (int** pp : res_i) {
        if ((r = dmalloc(c, (void**)pp, 4 * n_atoms))) return r;
        CU_TRY(c, cudaMemsetAsync(*pp, 0, 4 * n_atoms, s));
    }
    float** res_f[] = {&e.at.res, &e.at.rho};
    for (float** pp : res_f) {
        if ((r = dmalloc(c, (void**)pp, 4 * n_atoms))) return r;
        CU_TRY(c, cudaMemsetAsync(*pp, 0, 4 * n_atoms, s));
    }
    e.at.dim = c->d_dim; e.at.pos = c->d_pos; e.at.nb = c->d_atom_nb;
    if ((r = dmalloc(c, (void**)&c->d_e_atom, 8 * n_atoms))) return r;
    CU_TRY(c, cudaMemsetAsync(c->d_e_atom, 0, 8 * n_atoms, s));
    if ((r = dmalloc(c, (void**)&c->d_q_atom, 8 * n_atoms))) return r;
    CU_TRY(c, cudaMemsetAsync(c->d_q_atom, 0, 8 * n_atoms, s));
    if (use_umma(c)) {
        if (!encode_tiled_fn()) return fail(c, NOLSM_ECUDA, "cuTensorMapEncodeTiled not available");
        std::vector<CUtensorMap> maps((size_t)S * NMAP);
        const __half* vec0 = (const __half*)c->ws + (long long)S * e.slotsz;
        for (int sl = 0; sl < S; ++sl) {
            for (int b = 0; b < NBUF; ++b) {
                const __half* base = (const __half*)c->ws + (long long)sl * e.slotsz + (long long)b * e.bufsz;
                if (!make_tmap_f16_64x64(&maps[(size_t)sl * NMAP + b], base, e.cap, e.ld))
                    return fail(c, NOLSM_ECUDA, "cuTensorMapEncodeTiled failed");
            }
            for (int v = 0; v < 3; ++v) {       // maps 5, 6: the slot's vector blocks; map 7: the shared start block
                const __half* base = vec0 + (v < 2 ? (long long)sl * 2 + v : (long long)S * 2) * ((long long)e.cap * VLD);
                if (!make_tmap_f16_64x64(&maps[(size_t)sl * NMAP + NBUF + v], base, e.cap, VLD, VLD))
                    return fail(c, NOLSM_ECUDA, "cuTensorMapEncodeTiled failed");
            }
        }
        {   // start block of the power iterations: +-1 from a fixed hash in the first NVC columns, zero elsewhere
            std::vector<__half> v0((size_t)e.cap * VLD, __float2half(0.f));
            for (int rr = 0; rr < e.cap; ++rr)
                for (int cc = 0; cc < NVC; ++cc) {
                    unsigned h = (unsigned)(rr * NVC + cc) * 2654435761u + 0x9E3779B9u;
                    h ^= h >> 15; h *= 0x2C1B3C6Du; h ^= h >> 12; h *= 0x297A2D39u; h ^= h >> 15;
                    v0[(size_t)rr * VLD + cc] = __float2half((h & 1u) ? 1.f : -1.f);
                }
            CU_TRY(c, cudaMemcpyAsync((void*)(vec0 + (long long)S * 2 * ((long long)e.cap * VLD)), v0.data(), v0.size() * 2, cudaMemcpyHostToDevice, s));
            CU_TRY(c, cudaStreamSynchronize(s));      // `v0` is a local
        }
        if ((r = dmalloc(c, (void**)&c->d_maps, maps.size() * sizeof(CUtensorMap)))) return r;
        CU_TRY(c, cudaMemcpyAsync(c->d_maps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, s));
        CU_TRY(c, cudaStreamSynchronize(s));      // `maps` is a local
    }
    r = c->opt.precision == NOLSM_PREC_FP32 ? set_smem_limits<float>(c) : set_smem_limits<__half>(c);
    if (r) return r;
    if (c->persist) {
        PEngine& pe = c->peng;
        pe = PEngine{};
        if ((r = dmalloc(c, (void**)&pe.slots, sizeof(PSlot) * S))) return r;
        if ((r = dmalloc(c, (void**)&pe.gclaim, 8 * S))) return r;
        if ((r = dmalloc(c, (void**)&pe.sclaim, 4 * S))) return r;
        if ((r = dmalloc(c, (void**)&pe.ctr, 8 * PC_LEN))) return r;
        if ((r = dmalloc(c, (void**)&c->d_abort, 16))) return r;
        if ((r = dmalloc(c, (void**)&pe.heavy, 16))) return r;
        if ((r = dmalloc(c, (void**)&pe.pcols, (size_t)S * e.cap * PCW * sizeof(float)))) return r;
        if ((r = dmalloc(c, (void**)&pe.parked, 4 * S))) return r;
        pe.S = S; pe.cap = e.cap; pe.ld = e.ld; pe.bufsz = e.bufsz; pe.slotsz = e.slotsz;
        pe.tol_inv = e.tol_inv; pe.tol_sign = e.tol_sign; pe.max_inv = e.max_inv; pe.max_sign = e.max_sign;
        // Block power iteration (16 vectors, Frobenius growth): the estimate creeps up on rho from below (dense spectrum
        // edge: 0.75-0.80 rho after 3 steps, 0.84-0.87 after 6, 0.91-0.94 after 12 on the synthetic workloads), and an
        // overestimate is cheap (a factor 1.3 costs 0.3 scaled sign steps; the Schulz start converges for any
        // rho_hat > rho / 2) while an underestimate beyond 1.155 / alpha flips signs: few steps, generous safety.
        pe.p_s = c->opt.power_iters_s > 0 ? c->opt.power_iters_s : getenv_int("NOLSM_POW_S", 3);
        pe.p_a = c->opt.power_iters_a > 0 ? c->opt.power_iters_a : getenv_int("NOLSM_POW_A", 6);
        pe.safety_s = pe.p_s >= 6 ? 1.05f : 1.3f;
        pe.safety_a = pe.p_a >= 12 ? 1.05f : pe.p_a >= 6 ? 1.25f : 1.45f;
        if (const char* v = getenv("NOLSM_SAFETY_A")) pe.safety_a = (float)atof(v);
        pe.gather_rowatoms = g_rowatoms;
        {   // scaled Newton-Schulz schedule (C-6b): k0 steps with alpha_f, then the two optimal scalings
            // alpha = sqrt(3 / (1 + l + l^2)) for the interval [l, 1] the steps before leave the spectrum in
            const int k0 = c->opt.sign_scaled_iters;
            pe.n_sched = 0;
            if (k0 > 0) {
                const double af = c->opt.sign_scale;
                for (int k = 0; k < k0; ++k) pe.alpha_sched[pe.n_sched++] = (float)af;
                double l = 0.5 * af * (3.0 - af * af);
                for (int k = 0; k < 2; ++k) {
                    const double al = std::sqrt(3.0 / (1.0 + l + l * l));
                    pe.alpha_sched[pe.n_sched++] = (float)al;
                    l = 0.5 * al * l * (3.0 - al * al * l * l);
                }
            }
        }
        pe.ndie = (c->ndie == 2 && c->d_die && S >= 4) ? 2 : 1;
        pe.die_of_sm = c->d_die;
        pe.g_max = pe.ndie == 2 ? std::max(1, std::min(g_max, S) / 2) : std::max(1, std::min(g_max, S));
        pe.want_lead = std::max(1, getenv_int("NOLSM_WANT_LEAD", G2_WANT_LEAD));
        pe.dbg = getenv_int("NOLSM_DBG", 0);
        pe.gather_prefetch = getenv_int("NOLSM_GATHER_PREFETCH", 0);   // measured: no gain on cfg1 / cfg2, the loads in flight already cover the latency
        pe.split_tokens = getenv_int("NOLSM_SPLIT_TOKENS", 1);
        pe.half_tiles = c->opt.cluster_ctas == G4_CTAS ? 0 : getenv_int("NOLSM_HALF_TILES", 1);
        pe.tma_store = getenv_int("NOLSM_TMA_STORE", 1);
        pe.tile_n = getenv_int("NOLSM_TILE_N", BN) == 128 ? 128 : BN;
        pe.schulz_chunks = std::max(1, getenv_int("NOLSM_SCHULZ_CHUNKS", 16));
        pe.dcols_chunks = std::max(1, getenv_int("NOLSM_DCOLS_CHUNKS", 4));
        pe.next_atom = e.next_atom; pe.finished = e.finished; pe.abort_flag = c->d_abort;
        pe.at = e.at; pe.sv = sys_view(c);
        pe.udim = c->d_udim; pe.upos = c->d_upos; pe.adim = c->d_dim;
        pe.S_vals = c->dS; pe.H_vals = c->dH; pe.val_f64 = val_dtype == NOLSM_DTYPE_F64;
        pe.e_atom = c->d_e_atom; pe.q_atom = c->d_q_atom; pe.maps = c->d_maps; pe.base = (__half*)c->ws;
        c->h_sclaim0.assign(S, ((unsigned)SK_REFILL << 28) | (1u << 14));
        {   // every CTA waits on work published by the others: the whole grid must be resident at once
            const int ctas = c->opt.cluster_ctas == G4_CTAS ? G4_CTAS : 2;
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)(c->sms / ctas * ctas)); cfg.blockDim = dim3(P_THREADS); cfg.dynamicSmemBytes = P_SMEM_BYTES;
            cudaLaunchAttribute at;
            at.id = cudaLaunchAttributeClusterDimension;
            at.val.clusterDim.x = ctas; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
            cfg.attrs = &at; cfg.numAttrs = 1;
            int ncl = 0;
            if (ctas == G4_CTAS) CU_TRY(c, cudaOccupancyMaxActiveClusters(&ncl, nolsm_persist_kernel<G4_CTAS>, &cfg));
            else CU_TRY(c, cudaOccupancyMaxActiveClusters(&ncl, nolsm_persist_kernel<2>, &cfg));
            if (ncl < 1) return fail(c, NOLSM_ECUDA, "no cluster of the persistent kernel fits on this device");
            c->p_grid = ctas * std::min(ncl, c->sms / ctas);
            pe.ctas = ctas;
        }
        CU_TRY(c, cudaFuncSetAttribute(k_side_gather<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SIDE_SMEM));
        CU_TRY(c, cudaFuncSetAttribute(k_side_gather<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SIDE_SMEM));
    }
    CU_TRY(c, cudaStreamSynchronize(s));
    lap("workspace, maps, engine");
    c->assembled = true;
    return NOLSM_OK;
}

int nolsm_density_matrix_range(nolsm_ctx* c, double mu, int64_t a0, int64_t a1, void* D_vals, int d_dtype,
                               double* e_partial_host, void* cuda_stream) {
    if (!c) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "nolsm_assemble has not been called");
    if (!D_vals || a0 < 0 || a1 > c->n_atoms || a0 >= a1) return fail(c, NOLSM_EINVAL, "bad range or null D_vals");
    if (d_dtype != NOLSM_DTYPE_F64 && d_dtype != NOLSM_DTYPE_F32) return fail(c, NOLSM_EINVAL, "bad d_dtype");
    cudaStream_t us = (cudaStream_t)cuda_stream;
    cudaStream_t s = c->s_main;
    cudaSetDevice(c->dev);
    int r;
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
    // the engine runs on the library's own streams (the caller's stream may be the legacy default
    // stream, which cannot be captured); order them after the caller's stream
    CU_TRY(c, cudaEventRecord(c->ev_in, us));
    CU_TRY(c, cudaStreamWaitEvent(s, c->ev_in, 0));
    CU_TRY(c, cudaMemsetAsync(D_dev + (size_t)v0 * ds, 0, (size_t)(v1 - v0) * ds, s));
    CU_TRY(c, cudaMemsetAsync(c->d_e_atom + a0, 0, 8 * (a1 - a0), s));
    CU_TRY(c, cudaMemsetAsync(c->d_q_atom + a0, 0, 8 * (a1 - a0), s));
    c->ev_used = 0; c->recs.clear(); c->launches = 0; c->prof_on = false;
    c->last_persist = c->persist;
    if (c->persist) {
        // ---- persistent engine: one kernel launch evaluates the whole range ----
        PEngine pe = c->peng;
        // the feed counts units. Combined: every unit with a member in [a0, a1) is evaluated and serves its members inside
        // the range (a unit that straddles a range boundary is evaluated once per range it touches)
        int64_t u0 = a0, u1 = a1;
        if (c->combined) {
            c->h_feed.clear();
            std::vector<char> seen(c->n_units, 0);
            for (int64_t a = a0; a < a1; ++a) {
                const int32_t u = c->unit_of[a];
                if (!seen[u]) { seen[u] = 1; c->h_feed.push_back(u); }
            }
            std::sort(c->h_feed.begin(), c->h_feed.end());
            CU_TRY(c, cudaMemcpyAsync(c->d_feed, c->h_feed.data(), 4 * c->h_feed.size(), cudaMemcpyHostToDevice, s));
            u0 = 0; u1 = (int64_t)c->h_feed.size();
        }
        pe.mu = (float)mu; pe.a_end = (int)u1; pe.total = (int)(u1 - u0);
        pe.feed = c->combined ? c->d_feed : nullptr; pe.atom_lo = (int)a0; pe.atom_hi = (int)a1;
        pe.D_vals = D_dev; pe.d_f64 = d_dtype == NOLSM_DTYPE_F64;
        c->h_a0 = (int)u0;
        memset(c->h_ctr0, 0, sizeof(c->h_ctr0));
        c->h_ctr0[PC_T_START] = ~0ull;
        CU_TRY(c, cudaMemsetAsync(pe.slots, 0, sizeof(PSlot) * pe.S, s));
        CU_TRY(c, cudaMemsetAsync(pe.gclaim, 0, 8 * pe.S, s));
        CU_TRY(c, cudaMemcpyAsync(pe.sclaim, c->h_sclaim0.data(), 4 * pe.S, cudaMemcpyHostToDevice, s));
        CU_TRY(c, cudaMemcpyAsync(pe.ctr, c->h_ctr0, 8 * PC_LEN, cudaMemcpyHostToDevice, s));
        CU_TRY(c, cudaMemcpyAsync(pe.next_atom, &c->h_a0, 4, cudaMemcpyHostToDevice, s));
        CU_TRY(c, cudaMemsetAsync(pe.finished, 0, 4, s));
        CU_TRY(c, cudaMemsetAsync(c->d_abort, 0, 4, s));
        CU_TRY(c, cudaMemsetAsync(pe.heavy, 0, 8, s));
        CU_TRY(c, cudaMemsetAsync(pe.parked, 0, 4 * pe.S, s));
        CU_TRY(c, cudaEventRecord(c->ev_k0, s));
        {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)c->p_grid); cfg.blockDim = dim3(P_THREADS); cfg.dynamicSmemBytes = P_SMEM_BYTES; cfg.stream = s;
            cudaLaunchAttribute at;
            at.id = cudaLaunchAttributeClusterDimension;
            at.val.clusterDim.x = pe.ctas; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
            cfg.attrs = &at; cfg.numAttrs = 1;
            if (pe.ctas == G4_CTAS) CU_TRY(c, cudaLaunchKernelEx(&cfg, nolsm_persist_kernel<G4_CTAS>, pe));
            else CU_TRY(c, cudaLaunchKernelEx(&cfg, nolsm_persist_kernel<2>, pe));
        }
        CU_TRY(c, cudaGetLastError());
        CU_TRY(c, cudaEventRecord(c->ev_k1, s));
        c->launches = 1;
        c->rounds = 0;
        if (host_out) CU_TRY(c, cudaMemcpyAsync((char*)D_vals + (size_t)v0 * ds, c->d_D_stage, (size_t)(v1 - v0) * ds, cudaMemcpyDeviceToHost, s));
        CU_TRY(c, cudaEventRecord(c->ev_out, s));
        CU_TRY(c, cudaStreamWaitEvent(us, c->ev_out, 0));
        c->last_stream = us; c->last_a0 = a0; c->last_a1 = a1; c->have_result = true;
        if (e_partial_host) return nolsm_energy(c, e_partial_host);
        return NOLSM_OK;
    }
    Engine e = c->eng;
    e.mu = (float)mu;
    e.a_end = (int)a1;
    e.profiling = 0;
    const int a0i = (int)a0;
    CU_TRY(c, cudaMemsetAsync(e.slots, 0, sizeof(Slot) * e.S, s));
    CU_TRY(c, cudaMemcpyAsync(e.next_atom, &a0i, 4, cudaMemcpyHostToDevice, s));
    CU_TRY(c, cudaMemsetAsync(e.finished, 0, 4, s));
    CU_TRY(c, cudaMemsetAsync(e.prof, 0, sizeof(double) * PF_LEN, s));
    CU_TRY(c, cudaStreamSynchronize(s));       // a0i is a local; also makes *h_done = 0 below race-free
    *c->h_done = 0;
    const bool fp32 = c->opt.precision == NOLSM_PREC_FP32;

    // ---- one round captured as a CUDA graph ----
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    int64_t launches_per_round = 0;
    if (c->use_graph) {
        cudaGraph_t g = nullptr;
        CU_TRY(c, cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal));
        // The three branches of a round (GEMMs | gather + power iteration | D columns) are captured one after the other:
        // with concurrent branches the round engine hung intermittently on submatrices of ~1900 dimensions (B200, CUDA
        // 12.9; the serial capture never did, 6 of 6 against 2 of 5). NOLSM_FORK=1 restores the concurrent branches.
        const bool fork = getenv_int("NOLSM_FORK", 0) != 0;
        r = fp32 ? enqueue_round<float>(c, e, D_dev, d_dtype, fork) : enqueue_round<__half>(c, e, D_dev, d_dtype, fork);
        cudaError_t ce = cudaStreamEndCapture(s, &g);
        if (r) { if (g) cudaGraphDestroy(g); return r; }
        if (ce != cudaSuccess) { c->err = std::string("stream capture: ") + cudaGetErrorString(ce); return NOLSM_ECUDA; }
        ce = cudaGraphInstantiate(&c->graph_exec, g, 0);
        cudaGraphDestroy(g);
        if (ce != cudaSuccess) { c->err = std::string("graph instantiate: ") + cudaGetErrorString(ce); return NOLSM_ECUDA; }
        launches_per_round = c->launches;
        c->launches = 0;
    }

    // ---- replay rounds until the device reports every atom finished ----
    const int64_t total = a1 - a0;
    const int64_t max_rounds = ((total + e.S - 1) / e.S + 2) * (int64_t)(e.max_inv + e.max_sign + 8);
    int64_t round = 0, graph_rounds = 0;
    for (;; ++round) {
        if (round >= ROUND_DEPTH) {
            CU_TRY(c, cudaEventSynchronize(c->ev_round[round % ROUND_DEPTH]));
            if (*(volatile int*)c->h_done >= total) break;
        }
        if (round > max_rounds) return fail(c, NOLSM_ECUDA, "engine did not terminate");
        const bool prof = c->opt.profile_every > 0 && (round % c->opt.profile_every) == c->opt.profile_every / 2;
        if (prof || !c->use_graph) {
            Engine ep = e;
            ep.profiling = prof ? 1 : 0;
            c->prof_on = prof;
            r = fp32 ? enqueue_round<float>(c, ep, D_dev, d_dtype, false) : enqueue_round<__half>(c, ep, D_dev, d_dtype, false);
            c->prof_on = false;
            if (r) return r;
        } else {
            CU_TRY(c, cudaGraphLaunch(c->graph_exec, s));
            ++graph_rounds;
        }
        CU_TRY(c, cudaEventRecord(c->ev_round[round % ROUND_DEPTH], s));
    }
    c->launches += graph_rounds * launches_per_round;
    c->rounds = round;
    if (host_out) CU_TRY(c, cudaMemcpyAsync((char*)D_vals + (size_t)v0 * ds, c->d_D_stage, (size_t)(v1 - v0) * ds, cudaMemcpyDeviceToHost, s));
    CU_TRY(c, cudaEventRecord(c->ev_out, s));
    CU_TRY(c, cudaStreamWaitEvent(us, c->ev_out, 0));
    c->last_stream = us; c->last_a0 = a0; c->last_a1 = a1; c->have_result = true;
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
    if (int r = wait_result(c)) return r;
    const int64_t n = c->last_a1 - c->last_a0;
    std::vector<double> e(n);
    const int64_t u0 = c->combined ? 0 : c->last_a0, nu = c->combined ? c->n_units : n;   // status words are per unit
    std::vector<int> st(nu);
    CU_TRY(c, cudaMemcpy(e.data(), c->d_e_atom + c->last_a0, 8 * n, cudaMemcpyDeviceToHost));
    CU_TRY(c, cudaMemcpy(st.data(), c->eng.at.status + u0, 4 * nu, cudaMemcpyDeviceToHost));
    double sum = 0;
    int bits = 0;
    for (int64_t i = 0; i < n; ++i) sum += e[i];
    if (c->combined) { for (int32_t u : c->h_feed) bits |= st[u]; }           // the units of the last call
    else for (int64_t u = 0; u < nu; ++u) bits |= st[u];
    *e_elec = sum;
    if (bits & ST_NOTSPD) return fail(c, NOLSM_ENOTSPD, "an S_sub inverse iteration failed (see nolsm_get_atom_stats)");
    if (bits & ST_NOCONV) return fail(c, NOLSM_ENOCONV, "a sign iteration hit max_sign_iters (see nolsm_get_atom_stats)");
    return NOLSM_OK;
}

int nolsm_electron_count(nolsm_ctx* c, double* n_elec, double* q_atom_out) {
    if (!c || !n_elec) return NOLSM_EINVAL;
    if (!c->have_result) return fail(c, NOLSM_ESTATE, "no density matrix has been computed");
    cudaSetDevice(c->dev);
    if (int r = wait_result(c)) return r;
    const int64_t n = c->last_a1 - c->last_a0;
    std::vector<double> q(n);
    CU_TRY(c, cudaMemcpy(q.data(), c->d_q_atom + c->last_a0, 8 * n, cudaMemcpyDeviceToHost));
    double sum = 0;
    for (int64_t i = 0; i < n; ++i) sum += q[i];
    *n_elec = sum;
    if (q_atom_out) memcpy(q_atom_out, q.data(), 8 * n);
    return NOLSM_OK;
}

int nolsm_find_mu(nolsm_ctx* c, double n_target, double mu_lo, double mu_hi, double tol_n, double tol_mu, int max_evals,
                  void* D_vals, int d_dtype, void* cuda_stream, double* mu_out, double* n_out, int* evals_out) {
    if (!c || !D_vals || !mu_out) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "nolsm_assemble has not been called");
    if (!(mu_lo < mu_hi) || !(tol_n >= 0) || !(tol_mu >= 0)) return fail(c, NOLSM_EINVAL, "need mu_lo < mu_hi and tolerances >= 0");
    if (max_evals <= 0) max_evals = 40;
    // N(mu) = Tr(D(mu) S) never decreases with mu (it counts the generalised eigenvalues of every submatrix below mu,
    // weighted by their share in the atom's columns): bisection. Every evaluation is one nolsm_density_matrix call;
    // D_vals holds the density matrix of the last evaluated mu on return, which is the mu reported.
    int evals = 0, rc_soft = NOLSM_OK;
    auto count = [&](double mu, double* n) -> int {
        int r = nolsm_density_matrix(c, mu, D_vals, d_dtype, cuda_stream);
        if (r) return r;
        ++evals;
        double e;
        r = nolsm_energy(c, &e);
        if (r == NOLSM_ENOCONV) { rc_soft = r; r = NOLSM_OK; }       // flagged matrices are still written (nolsm.h)
        if (r) return r;
        return nolsm_electron_count(c, n, nullptr);
    };
    double n_lo, n_hi, mu = mu_lo, n_mu = 0;
    int r;
    if ((r = count(mu_lo, &n_lo))) return r;
    if ((r = count(mu_hi, &n_hi))) return r;
    mu = mu_hi; n_mu = n_hi;
    if (n_lo - tol_n > n_target || n_hi + tol_n < n_target) {
        if (n_out) *n_out = n_hi;
        if (evals_out) *evals_out = evals;
        *mu_out = mu_hi;
        return fail(c, NOLSM_EINVAL, "nolsm_find_mu: the electron count is not bracketed by [mu_lo, mu_hi]");
    }
    while (evals < max_evals && std::fabs(n_mu - n_target) > tol_n && (mu_hi - mu_lo) > tol_mu) {
        mu = 0.5 * (mu_lo + mu_hi);
        if ((r = count(mu, &n_mu))) return r;
        if (n_mu < n_target) mu_lo = mu; else mu_hi = mu;
    }
    *mu_out = mu;
    if (n_out) *n_out = n_mu;
    if (evals_out) *evals_out = evals;
    if (rc_soft) return fail(c, rc_soft, "a sign iteration hit max_sign_iters during the mu search (see nolsm_get_atom_stats)");
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

int nolsm_get_group(nolsm_ctx* c, int64_t atom, int32_t* members_out, int32_t* n_members_inout, int32_t* set_out,
                    int32_t* n_set_inout, int32_t* dim_out) {
    if (!c || !n_members_inout || !n_set_inout) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    if (atom < 0 || atom >= c->n_atoms) return fail(c, NOLSM_EINVAL, "atom out of range");
    const int32_t u = c->unit_of[atom];
    const int64_t m0 = c->unit_ptr[u], nm = c->unit_ptr[u + 1] - m0, s0 = c->uset_ptr[u], ns = c->uset_ptr[u + 1] - s0;
    if (dim_out) *dim_out = c->udim[u];
    int rc = NOLSM_OK;
    if (members_out) {
        if (*n_members_inout < nm) rc = fail(c, NOLSM_EINVAL, "members_out too small");
        else memcpy(members_out, c->unit_mem.data() + m0, sizeof(int32_t) * nm);
    }
    if (set_out) {
        if (*n_set_inout < ns) rc = fail(c, NOLSM_EINVAL, "set_out too small");
        else memcpy(set_out, c->uset_atom.data() + s0, sizeof(int32_t) * ns);
    }
    *n_members_inout = (int32_t)nm;
    *n_set_inout = (int32_t)ns;
    return rc;
}

int nolsm_gather_submatrix(nolsm_ctx* c, int64_t atom, int which, int out_fp16, void* out_host) {
    if (!c || !out_host || (which != 0 && which != 1)) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    if (c->combined) return fail(c, NOLSM_ESTATE, "nolsm_gather_submatrix returns per-atom submatrices: assemble without combine");
    if (atom < 0 || atom >= c->n_atoms) return fail(c, NOLSM_EINVAL, "atom out of range");
    cudaSetDevice(c->dev);
    const size_t es = out_fp16 ? 2 : 4;
    if ((size_t)c->eng.slotsz * es > c->ws_bytes) return fail(c, NOLSM_ENOMEM, "workspace too small for an FP32 gather");
    if (c->persist && out_fp16) {
        // the gather task of the persistent engine, launched stand-alone for slot 0
        int* d_atom;
        CU_TRY(c, cudaMalloc((void**)&d_atom, 4));
        const int a32 = (int)atom;
        CU_TRY(c, cudaMemcpy(d_atom, &a32, 4, cudaMemcpyHostToDevice));
        const PEngine& pe = c->peng;
        const int nset = (int)(c->nset_ptr[atom + 1] - c->nset_ptr[atom]);
        dim3 grid((nset + pe.gather_rowatoms - 1) / pe.gather_rowatoms, 1);
        if (c->val_dtype == NOLSM_DTYPE_F64)
            k_side_gather<double><<<grid, P_SIDE_THREADS, P_SIDE_SMEM, c->s_main>>>(pe.sv, (const double*)c->dS, (const double*)c->dH, pe.base, pe.slotsz, pe.bufsz, pe.ld, d_atom, c->d_dim, nullptr);
        else
            k_side_gather<float><<<grid, P_SIDE_THREADS, P_SIDE_SMEM, c->s_main>>>(pe.sv, (const float*)c->dS, (const float*)c->dH, pe.base, pe.slotsz, pe.bufsz, pe.ld, d_atom, c->d_dim, nullptr);
        cudaError_t ce = cudaGetLastError();
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(c->s_main);
        const int n = c->dim[atom];
        if (ce == cudaSuccess)
            ce = cudaMemcpy2D(out_host, (size_t)n * 2, (const char*)c->ws + (size_t)which * pe.bufsz * 2, (size_t)pe.ld * 2,
                              (size_t)n * 2, n, cudaMemcpyDeviceToHost);
        cudaFree(d_atom);
        if (ce != cudaSuccess) { c->err = cudaGetErrorString(ce); return NOLSM_ECUDA; }
        return NOLSM_OK;
    }
    // a one-slot view of the engine with the slot forced into phase NEW
    Engine e = c->eng;
    e.S = 1;
    e.profiling = 0;
    Slot sl{};
    sl.atom = (int)atom; sl.n = c->dim[atom]; sl.n16 = (sl.n + 15) & ~15; sl.pos = c->pos[atom]; sl.nbi = c->atom_nb[atom];
    sl.phase = sl.snap = PH_NEW;
    Slot* d_sl;
    CU_TRY(c, cudaMalloc((void**)&d_sl, sizeof(Slot)));
    CU_TRY(c, cudaMemcpy(d_sl, &sl, sizeof(Slot), cudaMemcpyHostToDevice));
    e.slots = d_sl;
    int r;
    const int dflt_prec = c->opt.precision;
    if (out_fp16) { r = set_smem_limits<__half>(c); if (!r) r = launch_gather<__half>(c, e, c->max_nset, c->s_main); }
    else { r = set_smem_limits<float>(c); if (!r) r = launch_gather<float>(c, e, c->max_nset, c->s_main); }
    (void)dflt_prec;
    if (!r) {
        cudaError_t ce = cudaStreamSynchronize(c->s_main);
        if (ce == cudaSuccess)
            ce = cudaMemcpy2D(out_host, (size_t)sl.n * es, (const char*)c->ws + (size_t)which * e.bufsz * es,
                              (size_t)e.ld * es, (size_t)sl.n * es, sl.n, cudaMemcpyDeviceToHost);
        if (ce != cudaSuccess) { c->err = cudaGetErrorString(ce); r = NOLSM_ECUDA; }
    }
    cudaFree(d_sl);
    return r;
}

int nolsm_get_atom_stats(nolsm_ctx* c, int64_t a0, int64_t count, int32_t* dims, int32_t* inv_iters, int32_t* sign_iters,
                         int32_t* status, int32_t* gemms, float* residual, double* e_atom) {
    if (!c) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    if (a0 < 0 || count < 0 || a0 + count > c->n_atoms) return fail(c, NOLSM_EINVAL, "range");
    cudaSetDevice(c->dev);
    if (c->have_result) { if (int r = wait_result(c)) return r; }
    if (c->combined) {
        // results are per unit: every member reports its unit's iteration counts, status and residual; the GEMMs and
        // the unit's dimension are reported by the unit's first member only (sums over atoms stay sums over units)
        const int64_t nu = c->n_units;
        std::vector<int32_t> ui(nu), us(nu), ut(nu), ug(nu);
        std::vector<float> ur(nu);
        CU_TRY(c, cudaMemcpy(ui.data(), c->eng.at.inv, 4 * nu, cudaMemcpyDeviceToHost));
        CU_TRY(c, cudaMemcpy(us.data(), c->eng.at.sign, 4 * nu, cudaMemcpyDeviceToHost));
        CU_TRY(c, cudaMemcpy(ut.data(), c->eng.at.status, 4 * nu, cudaMemcpyDeviceToHost));
        CU_TRY(c, cudaMemcpy(ug.data(), c->eng.at.gemms, 4 * nu, cudaMemcpyDeviceToHost));
        CU_TRY(c, cudaMemcpy(ur.data(), c->eng.at.res, 4 * nu, cudaMemcpyDeviceToHost));
        for (int64_t k = 0; k < count; ++k) {
            const int64_t a = a0 + k;
            const int32_t u = c->unit_of[a];
            const bool first = c->unit_mem[c->unit_ptr[u]] == a;
            if (dims) dims[k] = first ? c->udim[u] : 0;
            if (inv_iters) inv_iters[k] = ui[u];
            if (sign_iters) sign_iters[k] = us[u];
            if (status) status[k] = ut[u];
            if (gemms) gemms[k] = first ? ug[u] : 0;
            if (residual) residual[k] = ur[u];
        }
        if (e_atom) CU_TRY(c, cudaMemcpy(e_atom, c->d_e_atom + a0, 8 * count, cudaMemcpyDeviceToHost));
        return NOLSM_OK;
    }
    if (dims) memcpy(dims, c->dim.data() + a0, 4 * count);
    if (inv_iters) CU_TRY(c, cudaMemcpy(inv_iters, c->eng.at.inv + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (sign_iters) CU_TRY(c, cudaMemcpy(sign_iters, c->eng.at.sign + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (status) CU_TRY(c, cudaMemcpy(status, c->eng.at.status + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (gemms) CU_TRY(c, cudaMemcpy(gemms, c->eng.at.gemms + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (residual) CU_TRY(c, cudaMemcpy(residual, c->eng.at.res + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (e_atom) CU_TRY(c, cudaMemcpy(e_atom, c->d_e_atom + a0, 8 * count, cudaMemcpyDeviceToHost));
    return NOLSM_OK;
}

int nolsm_get_stats(nolsm_ctx* c, nolsm_stats* out) {
    if (!c || !out) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    memset(out, 0, sizeof(*out));
    const int64_t n = c->n_atoms;
    out->n_atoms = n;
    out->n_batches = c->rounds;
    out->n_units = c->n_units;
    out->dim_min = 1 << 30;
    double dsum = 0;
    for (int64_t u = 0; u < c->n_units; ++u) {
        out->dim_min = std::min<int64_t>(out->dim_min, c->udim[u]);
        out->dim_max = std::max<int64_t>(out->dim_max, c->udim[u]);
        dsum += c->udim[u];
    }
    out->dim_mean = dsum / (double)c->n_units;
    if (c->have_result) {
        std::vector<int32_t> dm(n), inv(n), sg(n), st(n), gm(n);
        int r = nolsm_get_atom_stats(c, 0, n, dm.data(), inv.data(), sg.data(), st.data(), gm.data(), nullptr, nullptr);
        if (r) return r;
        for (int64_t i = c->last_a0; i < c->last_a1; ++i) {
            if (dm[i] == 0) continue;                       // not the first member of its unit
            out->sum_inv_iters += inv[i]; out->sum_sign_iters += sg[i]; out->gemms_executed += gm[i];
            const double d = dm[i];
            out->flops_useful += 2.0 * d * d * d * gm[i];
            int ntm, ntn;
            const int n16 = (dm[i] + 15) & ~15;
            choose_tiling(n16, ntm, ntn);
            // rows the tensor cores executed: 256 per row block; the persistent pair engine runs a last row block of at most
            // 128 rows as M = 128 tiles (except on a ragged last column tile whose width is not a multiple of 32)
            double rows = (double)(ntm * BM);
            if (c->last_persist && c->peng.half_tiles && n16 - (ntm - 1) * BM <= BM / 2) {
                const int last_bn = n16 - (ntn - 1) * BN;
                rows -= (BM / 2) * ((last_bn & 31) == 0 ? 1.0 : (double)(n16 - last_bn) / (double)n16);
            }
            out->flops_padded += 2.0 * rows * (double)n16 * (double)n16 * gm[i];
            out->n_notspd += (st[i] & ST_NOTSPD) ? 1 : 0;
            out->n_noconv += (st[i] & ST_NOCONV) ? 1 : 0;
        }
        const size_t es = elem_size(c), vs = c->val_dtype == NOLSM_DTYPE_F64 ? 8 : 4;
        for (int64_t i = c->last_a0; i < c->last_a1; ++i) {
            const double n16 = (dm[i] + 15) & ~15, n = c->dim[i];
            const double nv = (double)(c->blk_off[c->row_ptr[i + 1]] - c->blk_off[c->row_ptr[i]]);
            out->gather_bytes += 2.0 * n16 * n16 * es;                       // dense S_sub and H_sub written (once per unit)
            out->scatter_bytes += nv * (c->last_ds + vs) + (n * n + n * c->atom_nb[i]) * es;
        }
    }
    return NOLSM_OK;
}

int nolsm_get_profile(nolsm_ctx* c, double* out, int n) {
    if (!c || !out || n < NOLSM_PROFILE_LEN) return NOLSM_EINVAL;
    if (!c->have_result) return fail(c, NOLSM_ESTATE, "no density matrix has been computed");
    cudaSetDevice(c->dev);
    if (int r = wait_result(c)) return r;
    if (c->last_persist) {
        // one launch: the kernel's duration from CUDA events on its stream; side-task times are summed
        // over the side groups (SM-time, the tasks run concurrently with the GEMM pipeline)
        unsigned long long ct[PC_LEN];
        CU_TRY(c, cudaMemcpy(ct, c->peng.ctr, sizeof(ct), cudaMemcpyDeviceToHost));
        float kms = 0;
        CU_TRY(c, cudaEventElapsedTime(&kms, c->ev_k0, c->ev_k1));
        nolsm_stats st;
        if (int r = nolsm_get_stats(c, &st)) return r;
        out[0] = ct[PC_SIDE_NS + SK_GATHER] * 1e-6; out[1] = (double)ct[PC_SIDE_TASKS + SK_GATHER]; out[2] = (double)ct[PC_SIDE_BYTES + SK_GATHER];
        out[3] = kms; out[4] = 1; out[5] = st.flops_useful; out[6] = st.flops_padded;
        out[7] = ct[PC_SIDE_NS + SK_DCOLS] * 1e-6; out[8] = (double)ct[PC_SIDE_TASKS + SK_DCOLS]; out[9] = (double)ct[PC_SIDE_BYTES + SK_DCOLS];
        out[10] = (ct[PC_SIDE_NS + SK_REFILL] + ct[PC_SIDE_NS + SK_SCHULZ1]) * 1e-6;
        out[11] = (double)(ct[PC_SIDE_TASKS + SK_REFILL] + ct[PC_SIDE_TASKS + SK_SCHULZ1]);
        out[12] = (double)(c->last_a1 - c->last_a0); out[13] = 1;
        return NOLSM_OK;
    }
    double ms[4] = {0, 0, 0, 0}, cnt[4] = {0, 0, 0, 0};
    for (const nolsm_ctx::Rec& r : c->recs) {
        float t = 0;
        if (cudaEventElapsedTime(&t, c->ev_pool[r.ev], c->ev_pool[r.ev + 1]) != cudaSuccess) { cudaGetLastError(); continue; }
        ms[r.kind] += t; cnt[r.kind] += 1;
    }
    double pf[PF_LEN];
    CU_TRY(c, cudaMemcpy(pf, c->eng.prof, sizeof(pf), cudaMemcpyDeviceToHost));
    const size_t es = elem_size(c), vs = c->val_dtype == NOLSM_DTYPE_F64 ? 8 : 4;
    out[0] = ms[K_GATHER]; out[1] = cnt[K_GATHER]; out[2] = pf[PF_GATHER_SRC] * vs + pf[PF_GATHER_DENSE] * es;
    out[3] = ms[K_GEMM]; out[4] = cnt[K_GEMM]; out[5] = pf[PF_FLOP_USEFUL]; out[6] = pf[PF_FLOP_PADDED];
    out[7] = ms[K_DCOLS]; out[8] = cnt[K_DCOLS]; out[9] = pf[PF_DCOLS_BYTES];
    out[10] = ms[K_OTHER]; out[11] = cnt[K_OTHER];
    out[12] = pf[PF_SUBMATS]; out[13] = (double)c->launches;
    return NOLSM_OK;
}

int nolsm_get_engine_counters(nolsm_ctx* c, double* out, int n) {
    if (!c || !out || n < NOLSM_COUNTERS_LEN) return NOLSM_EINVAL;
    if (!c->have_result) return fail(c, NOLSM_ESTATE, "no density matrix has been computed");
    for (int i = 0; i < NOLSM_COUNTERS_LEN; ++i) out[i] = 0;
    if (!c->last_persist) return NOLSM_OK;
    cudaSetDevice(c->dev);
    if (int r = wait_result(c)) return r;
    unsigned long long ct[PC_LEN];
    CU_TRY(c, cudaMemcpy(ct, c->peng.ctr, sizeof(ct), cudaMemcpyDeviceToHost));
    float kms = 0;
    CU_TRY(c, cudaEventElapsedTime(&kms, c->ev_k0, c->ev_k1));
#ifdef NOLSM_TIMING
    {
        unsigned long long t[16];
        cudaMemcpyFromSymbol(t, g4_timing, sizeof(t));
        static const char* nm[16] = {"mma_take", "mma_tempty", "mma_full", "mma_total", "epi_take", "epi_tfull(cum)", "epi_work(cum)", "epi_done(cum)",
                                     "prod_empty", "prod_total", "prod_take", "mma_fulltile_cyc", "mma_fulltiles", "", "", ""};
        for (int i = 0; i < 13; ++i) fprintf(stderr, "g4_timing %-16s %.3f Gcyc\n", nm[i], t[i] * 1e-9);
        fprintf(stderr, "gather phases (thread 0 of every side group, Gcyc): lookup %.3f zero %.3f stream %.3f writeout %.3f\n", t[12] * 1e-9, t[13] * 1e-9, t[14] * 1e-9, t[15] * 1e-9);
        if (t[12]) fprintf(stderr, "g4_timing cycles per full-width tile (tempty wait + k-loop): %.0f\n", (double)t[11] / (double)t[12]);
        unsigned long long z[16] = {};
        cudaMemcpyToSymbol(g4_timing, z, sizeof(z));
#ifdef G2_TIMING
        unsigned long long t2[12];
        cudaMemcpyFromSymbol(t2, g2_timing, sizeof(t2));
        if (t2[9]) fprintf(stderr, "g2_timing cycles per full-width tile (tempty wait + k-loop): %.0f over %.0f tiles\n", (double)t2[8] / (double)t2[9], (double)t2[9]);
        static const char* nm2[8] = {"mma_take", "mma_tempty", "mma_full", "mma_total", "epi_take", "epi_tfull", "epi_work(cum)", "epi_done(cum)"};
        for (int i = 0; i < 8; ++i) fprintf(stderr, "g2_timing %-16s %.3f Gcyc\n", nm2[i], t2[i] * 1e-9);
        cudaMemcpyToSymbol(g2_timing, z, sizeof(t2));
#endif
    }
#endif
    out[0] = 1; out[1] = kms; out[2] = (double)(ct[PC_T_END] - ct[PC_T_START]) * 1e-6;
    out[3] = (double)ct[PC_TILES]; out[4] = ct[PC_SCHED_IDLE_NS] * 1e-6; out[5] = ct[PC_SCHED_BUSY_NS] * 1e-6;
    out[6] = (double)ct[PC_OVERSHOOT]; out[7] = c->peng.S; out[8] = c->p_grid / 2;
    for (int k = 0; k < 8; ++k) {
        out[9 + k] = ct[PC_SIDE_NS + k] * 1e-6;
        out[17 + k] = (double)ct[PC_SIDE_BYTES + k];
        out[25 + k] = (double)ct[PC_SIDE_TASKS + k];
    }
    return NOLSM_OK;
}

}  // extern "C"
