// Host-side context of the NOLSM library (include/nolsm.h) and the helpers its translation units share:
//   abi.cpp      context life cycle, results, diagnostics
//   assemble.cpp nolsm_assemble: validation, index sets N(i), workspace plan, tensor maps         (a0)
//   grouping.cpp submatrix combination: Eq. 9 / Eq. 10 costs, greedy groups
//   engine.cu    the launches: persistent kernel (a1-a7), round engine (FP32 validation), stand-alone side tasks
#pragma once
#include <algorithm>
#include <chrono>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <exception>
#include <new>
#include <system_error>
#include <string>
#include <thread>
#include <vector>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/nolsm.h"

namespace nolsm {
struct Engine;
struct PEngine;
}

constexpr int NOLSM_ROUND_DEPTH = 4;    // rounds kept in flight ahead of the device (round engine)
constexpr int NOLSM_MAX_MU = 8;         // == P_MAX_MU (persist.cuh)
constexpr int NOLSM_ABORT_HIST = 16;    // abort words of earlier launches kept until a call waits for the results

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
    // p(n) of Eq. 10: measured multiplication rate at dimensions pn_n (ascending), in GFLOP/s (integers)
    std::vector<int64_t> pn_n, pn_rate;

    // device arrays
    std::vector<std::pair<void*, size_t>> owned;   // everything cudaMalloc'ed by assemble
    std::vector<std::pair<void*, size_t>> pool;    // blocks of the previous assemble, reused by the next one (cudaFree of GB-sized
                                                   // blocks stalled re-assembly for up to 0.7 s; freed by nolsm_destroy)
    long long *d_row_ptr = nullptr, *d_blk_off = nullptr, *d_nset_ptr = nullptr;
    int *d_col_idx = nullptr, *d_atom_nb = nullptr, *d_nset_atom = nullptr, *d_nset_slot = nullptr, *d_nset_off = nullptr;
    const void *dH = nullptr, *dS = nullptr;
    int val_dtype = NOLSM_DTYPE_F64;

    // engine (nolsm_device.cuh / persist.cuh): the structs live in engine.cu's view; here they are opaque blobs
    nolsm::Engine* eng = nullptr;
    nolsm::PEngine* peng = nullptr;
    void* ws = nullptr;
    size_t ws_bytes = 0;
    CUtensorMap* d_maps = nullptr;
    float *d_vec = nullptr, *d_nrm = nullptr;
    int* h_done = nullptr;              // pinned, mapped
    int *d_dim = nullptr, *d_pos = nullptr;
    double* d_e_atom = nullptr;
    double* d_q_atom = nullptr;
    double* d_mu_acc = nullptr;         // [2 * NOLSM_MAX_MU] electron counts and energies per trial mu (nolsm_electron_counts)
    int* d_gsym = nullptr;              // [n_units] symmetric GEMMs per unit
    cudaStream_t s_main = nullptr, s_x = nullptr;
    cudaEvent_t ev_in = nullptr, ev_out = nullptr;
    cudaEvent_t ev_round[NOLSM_ROUND_DEPTH] = {};
    cudaGraphExec_t graph_exec = nullptr;
    bool use_graph = true;

    // persistent engine (persist.cuh): one kernel launch per density_matrix call
    bool persist = false;
    int* d_abort = nullptr;             // [1 + NOLSM_ABORT_HIST]: the running kernel's abort word, then the final words of the
                                        // launches nobody has waited for yet (launch k at 1 + k % NOLSM_ABORT_HIST)
    int64_t launch_seq = 0, checked_seq = 0;   // persistent launches since assemble; launches whose abort word has been read
    std::chrono::steady_clock::time_point t_launch{};   // when the last persistent kernel was enqueued (host time limit)
    unsigned long long h_stall_ns = 0;  // device watchdog limit of the hot waits, from timeout_s
    // D of a call with pageable host output stays in d_D_stage until a call waits for the result (wait_result copies it)
    void* pend_dst = nullptr;
    size_t pend_bytes = 0;
    int p_grid = 0;                     // CTAs of the persistent kernel
    cudaEvent_t ev_k0 = nullptr, ev_k1 = nullptr;
    int h_a0 = 0;
    std::vector<unsigned long long> h_ctr0;
    std::vector<unsigned int> h_sclaim0;
    bool last_persist = false;
    double timeout_s = 300.0;
    int n_mu_last = 1;                  // trial mu of the last call
    bool last_count_only = false;

    // last density call
    cudaStream_t last_stream = nullptr;
    int64_t last_a0 = 0, last_a1 = 0;
    bool have_result = false;
    void* d_D_stage = nullptr;
    size_t d_D_stage_bytes = 0;
    size_t last_ds = 8;
    int64_t rounds = 0;

    // sampled per-launch profiling of the round engine (options.profile_every): CUDA events on the launching stream
    struct Rec { int kind; size_t ev; };
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    std::vector<Rec> recs;
    bool prof_on = false;
    int64_t launches = 0;
};

#define CU_TRY(ctx, expr)                                                                           \
    do {                                                                                            \
        cudaError_t e_ = (expr);                                                                    \
        if (e_ != cudaSuccess) {                                                                    \
            (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(e_);                       \
            return e_ == cudaErrorMemoryAllocation ? NOLSM_ENOMEM : NOLSM_ECUDA;                   \
        }                                                                                           \
    } while (0)

namespace nolsm_host {

// f(begin, end) over chunks of [0, n) on up to 16 threads. An exception inside a worker (std::bad_alloc of a per-thread
// vector) is carried to the caller and rethrown there after every worker has been joined; if a thread cannot be
// started, the caller's thread does that chunk itself.
template <typename F>
void parallel_for(int64_t n, F f) {
    unsigned nt = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
    if (n < 1 << 11) nt = 1;
    if (nt == 1) { f(0, n); return; }
    std::vector<std::thread> th;
    std::vector<std::exception_ptr> err(nt);
    th.reserve(nt);
    const int64_t chunk = (n + nt - 1) / nt;
    for (unsigned t = 0; t < nt; ++t) {
        const int64_t b = t * chunk, e = std::min<int64_t>(n, b + chunk);
        if (b >= e) continue;
        auto work = [&f, &err, t, b, e] { try { f(b, e); } catch (...) { err[t] = std::current_exception(); } };
        try { th.emplace_back(work); } catch (const std::system_error&) { work(); }
    }
    for (auto& x : th) x.join();
    for (auto& ep : err) if (ep) std::rethrow_exception(ep);
}

// Temporary device buffers and events of the diagnostics: released on every return path.
struct DevBuf {
    void* p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    template <typename T> T* as() const { return static_cast<T*>(p); }
};
struct EventPair {
    cudaEvent_t a = nullptr, b = nullptr;
    ~EventPair() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); }
};

inline int fail(nolsm_ctx* c, int code, const std::string& msg) { c->err = msg; return code; }
// Handler of the function-try-block around every extern "C" entry point: no exception crosses the C boundary
// (std::bad_alloc from the host-side vectors, std::system_error from the worker threads of parallel_for).
inline int on_exception(nolsm_ctx* c, const char* where) {
    int code = NOLSM_ENOMEM;
    std::string what = "out of host memory";
    try { throw; }
    catch (const std::bad_alloc&) {}
    catch (const std::exception& e) { code = NOLSM_ECUDA; what = e.what(); }
    catch (...) { code = NOLSM_ECUDA; what = "unknown exception"; }
    if (c) { try { c->err = std::string(where) + ": " + what; } catch (...) {} }
    return code;
}
inline bool verbose(int level = 1) {
    static const int v = [] { const char* s = getenv("NOLSM_VERBOSE"); return s && *s ? atoi(s) : 0; }();
    return v >= level;
}

// abi.cpp
bool is_device_ptr(const void* p);
int dmalloc(nolsm_ctx* c, void** p, size_t bytes);
void free_assembled(nolsm_ctx* c, bool release = false);
int to_device(nolsm_ctx* c, const void* src, size_t bytes, const void** out, cudaStream_t s);
int to_host(nolsm_ctx* c, const void* src, size_t bytes, void* dst, cudaStream_t s);
int wait_result(nolsm_ctx* c);
int check_abort_words(nolsm_ctx* c);    // reads the abort words of every launch since the last check
inline size_t elem_size(const nolsm_ctx* c) { return c->opt.precision == NOLSM_PREC_FP32 ? 4 : 2; }
inline bool use_umma(const nolsm_ctx* c) { return c->opt.precision != NOLSM_PREC_FP32 && c->opt.gemm_backend != NOLSM_GEMM_SIMT; }
// The persistent engine serves the mixed-precision tcgen05 path; the round engine (plain FFMA GEMMs) serves the FP32
// validation mode and gemm_backend = SIMT.
inline bool want_persist(const nolsm_ctx* c) { return use_umma(c) && c->opt.engine != NOLSM_ENGINE_ROUNDS; }

// grouping.cpp
int64_t combine_cost(const nolsm_ctx* c, int64_t n, int mode);
void build_units(nolsm_ctx* c, int mode, int max_dim, int max_members, int max_cand);

// engine.cu
int engine_create(nolsm_ctx* c);                      // kernel attributes (once per context)
void engine_destroy(nolsm_ctx* c);
int engine_plan(nolsm_ctx* c, cudaStream_t s);        // slots, workspace, tensor maps, engine parameter blocks (end of assemble)
int engine_block_keep(nolsm_ctx* c, unsigned char* d_keep, cudaStream_t s);     // C-1 filter kernel
int engine_run(nolsm_ctx* c, const double* mu, int n_mu, bool count_only, int64_t a0, int64_t a1, char* D_dev, int d_dtype, cudaStream_t s);
int engine_stats(nolsm_ctx* c, nolsm_stats* out);
int engine_profile(nolsm_ctx* c, double* out);
int engine_counters(nolsm_ctx* c, double* out);
int engine_atom_stats(nolsm_ctx* c, int64_t a0, int64_t count, int32_t* dims, int32_t* inv_iters, int32_t* sign_iters,
                      int32_t* status, int32_t* gemms, float* residual, double* e_atom);
int engine_status_bits(nolsm_ctx* c, int* bits);
int engine_gather(nolsm_ctx* c, int64_t unit_or_atom, bool is_unit, int which, int out_fp16, void* out_host);
int engine_side_bandwidth(nolsm_ctx* c, int which, int reps, double* ms_out, double* bytes_out);
int engine_gather_noalloc(nolsm_ctx* c, int64_t unit, int which, void* out, cudaStream_t s);   // static device scratch, no allocation

}  // namespace nolsm_host
