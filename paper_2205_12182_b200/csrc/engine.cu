// Everything of the NOLSM library that launches kernels: the workspace plan of nolsm_assemble (slots, tensor maps,
// engine parameter blocks), the persistent kernel of the mixed-precision path (persist.cuh: a1-a7 of a call in ONE
// launch), the round engine of the FP32 validation mode (kernels.cuh: plain FFMA GEMMs, one CUDA graph per iteration
// round), the stand-alone side-task launches (gather / scatter bandwidth), and the results the kernels leave on the device.
#include <cmath>

#include "ctx.h"
#include "kernels.cuh"
#include "persist.cuh"
#include "tmap_host.h"

using namespace nolsm;
using namespace nolsm_host;

namespace {

enum { K_GATHER = 0, K_GEMM = 1, K_DCOLS = 2, K_OTHER = 3 };

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

SysView sys_view(const nolsm_ctx* c) {
    SysView v;
    v.row_ptr = c->d_row_ptr; v.col_idx = c->d_col_idx; v.blk_off = c->d_blk_off; v.atom_nb = c->d_atom_nb;
    v.nset_ptr = c->d_nset_ptr; v.nset_atom = c->d_nset_atom; v.nset_slot = c->d_nset_slot; v.nset_off = c->d_nset_off;
    v.unit_ptr = c->d_unit_ptr; v.unit_mem = c->d_unit_mem; v.uset_ptr = c->d_uset_ptr; v.uset_atom = c->d_uset_atom;
    v.uset_off = c->d_uset_off; v.nset_uoff = c->d_nset_uoff;
    return v;
}

// ---------------------------------------------------------------------------------------------------------------
// Round engine (FP32 validation mode / SIMT GEMMs)
// ---------------------------------------------------------------------------------------------------------------
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
    const int t64 = (e.cap + 63) / 64;
    LAUNCH(c, K_GEMM, s, k_gemm_simt<T><<<dim3(t64 * t64, e.S), 256, 0, s>>>(e, (T*)c->ws, launch));
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
    const int g = (int)std::max<size_t>(gather_smem(c->max_nset, c->eng->cap), 48 * 1024);
    const int d = (int)std::max<size_t>(dcols_smem(c), 48 * 1024);
    if (d > 227 * 1024 || g > 227 * 1024) return fail(c, NOLSM_EINVAL, "index set or n_i * nb(i) too large for the round engine's kernels");
    CU_TRY(c, cudaFuncSetAttribute(k_gather<double, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, g));
    CU_TRY(c, cudaFuncSetAttribute(k_gather<float, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, g));
    CU_TRY(c, cudaFuncSetAttribute(k_dcols_scatter<T, double, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, d));
    CU_TRY(c, cudaFuncSetAttribute(k_dcols_scatter<T, double, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, d));
    CU_TRY(c, cudaFuncSetAttribute(k_dcols_scatter<T, float, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, d));
    CU_TRY(c, cudaFuncSetAttribute(k_dcols_scatter<T, float, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, d));
    return NOLSM_OK;
}

// One round (nolsm_device.cuh), all kernels on one stream: round begin, D columns of the slots in phase FIN, gather and
// power iterations of the slots in phase NEW / PA, the two grouped GEMM launches.
template <typename T>
int enqueue_round(nolsm_ctx* c, const Engine& e, void* D, int d_dtype) {
    cudaStream_t sm = c->s_main;
    LAUNCH(c, K_OTHER, sm, k_round_begin<<<1, MAX_SLOTS, 0, sm>>>(e));
    if (d_dtype == NOLSM_DTYPE_F64) launch_dcols<T, double>(c, e, (double*)D, sm);
    else launch_dcols<T, float>(c, e, (float*)D, sm);
    int r;
    if ((r = launch_gather<T>(c, e, c->max_nset, sm))) return r;
    const int P = std::max(e.p_s, e.p_a);
    LAUNCH(c, K_OTHER, sm, k_vec_init<<<dim3((e.cap + 255) / 256, e.S), 256, 0, sm>>>(e, c->d_vec, c->d_nrm, P));
    for (int it = 0; it < P; ++it)
        LAUNCH(c, K_OTHER, sm, k_matvec<T><<<dim3(16, e.S), 256, 0, sm>>>(e, (const T*)c->ws, c->d_vec, c->d_nrm, it));
    LAUNCH(c, K_OTHER, sm, k_power_finish<T><<<dim3(32, e.S), 256, 0, sm>>>(e, (T*)c->ws, c->d_nrm));
    launch_gemm<T>(c, e, 0, sm);
    launch_gemm<T>(c, e, 1, sm);
    CU_TRY(c, cudaGetLastError());
    return NOLSM_OK;
}

int run_rounds(nolsm_ctx* c, double mu, int64_t a0, int64_t a1, char* D_dev, int d_dtype) {
    cudaStream_t s = c->s_main;
    Engine e = *c->eng;
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
    int r;

    // ---- one round captured as a CUDA graph ----
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    int64_t launches_per_round = 0;
    if (c->use_graph) {
        cudaGraph_t g = nullptr;
        CU_TRY(c, cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal));
        r = fp32 ? enqueue_round<float>(c, e, D_dev, d_dtype) : enqueue_round<__half>(c, e, D_dev, d_dtype);
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
        if (round >= NOLSM_ROUND_DEPTH) {
            CU_TRY(c, cudaEventSynchronize(c->ev_round[round % NOLSM_ROUND_DEPTH]));
            if (*(volatile int*)c->h_done >= total) break;
        }
        if (round > max_rounds) return fail(c, NOLSM_ECUDA, "engine did not terminate");
        const bool prof = c->opt.profile_every > 0 && (round % c->opt.profile_every) == c->opt.profile_every / 2;
        if (prof || !c->use_graph) {
            Engine ep = e;
            ep.profiling = prof ? 1 : 0;
            c->prof_on = prof;
            r = fp32 ? enqueue_round<float>(c, ep, D_dev, d_dtype) : enqueue_round<__half>(c, ep, D_dev, d_dtype);
            c->prof_on = false;
            if (r) return r;
        } else {
            CU_TRY(c, cudaGraphLaunch(c->graph_exec, s));
            ++graph_rounds;
        }
        CU_TRY(c, cudaEventRecord(c->ev_round[round % NOLSM_ROUND_DEPTH], s));
    }
    c->launches += graph_rounds * launches_per_round;
    c->rounds = round;
    return NOLSM_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// Persistent engine
// ---------------------------------------------------------------------------------------------------------------
int run_persistent(nolsm_ctx* c, const double* mu, int n_mu, bool count_only, int64_t a0, int64_t a1, char* D_dev, int d_dtype) {
    cudaStream_t s = c->s_main;
    PEngine pe = *c->peng;
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
    pe.n_mu = n_mu;
    for (int j = 0; j < n_mu; ++j) pe.mu[j] = (float)mu[j];
    pe.count_only = count_only ? 1 : 0;
    pe.a_end = (int)u1; pe.total = (int)(u1 - u0);
    pe.feed = c->combined ? c->d_feed : nullptr; pe.atom_lo = (int)a0; pe.atom_hi = (int)a1;
    pe.D_vals = D_dev; pe.d_f64 = d_dtype == NOLSM_DTYPE_F64;
    c->h_a0 = (int)u0;
    c->h_ctr0.assign(PC_LEN, 0ull);
    c->h_ctr0[PC_T_START] = ~0ull;
    CU_TRY(c, cudaMemsetAsync(pe.slots, 0, sizeof(PSlot) * pe.S, s));
    CU_TRY(c, cudaMemsetAsync(pe.gclaim, 0, 8 * pe.S, s));
    CU_TRY(c, cudaMemcpyAsync(pe.sclaim, c->h_sclaim0.data(), 4 * pe.S, cudaMemcpyHostToDevice, s));
    CU_TRY(c, cudaMemcpyAsync(pe.ctr, c->h_ctr0.data(), 8 * PC_LEN, cudaMemcpyHostToDevice, s));
    CU_TRY(c, cudaMemcpyAsync(pe.next_atom, &c->h_a0, 4, cudaMemcpyHostToDevice, s));
    CU_TRY(c, cudaMemsetAsync(pe.finished, 0, 4, s));
    // the abort word of the previous launch is kept (stream order: after that kernel) before this launch clears it; when
    // the history is full the host waits and reads it first
    if (c->launch_seq - c->checked_seq >= NOLSM_ABORT_HIST) {
        CU_TRY(c, cudaStreamSynchronize(s));
        if (int r = check_abort_words(c)) return r;
    }
    if (c->launch_seq > c->checked_seq)
        CU_TRY(c, cudaMemcpyAsync(c->d_abort + 1 + (c->launch_seq - 1) % NOLSM_ABORT_HIST, c->d_abort, 4, cudaMemcpyDeviceToDevice, s));
    CU_TRY(c, cudaMemsetAsync(c->d_abort, 0, 4, s));
    // device watchdog from options.timeout_s: a hot wait (k-loop stages, accumulators) may last timeout_s / 10, an idle
    // wait (tile records, ring entries: ten rounds of that) timeout_s
    c->h_stall_ns = (unsigned long long)(std::max(2.0, c->timeout_s / 10.0) * 1e9);
    CU_TRY(c, cudaMemcpyToSymbolAsync(g_stall_ns, &c->h_stall_ns, 8, 0, cudaMemcpyHostToDevice, s));
    CU_TRY(c, cudaMemsetAsync(pe.heavy, 0, 8, s));
    CU_TRY(c, cudaMemsetAsync(pe.parked, 0, 4 * pe.S, s));
    CU_TRY(c, cudaMemsetAsync(c->d_mu_acc, 0, 16 * NOLSM_MAX_MU, s));
    CU_TRY(c, cudaEventRecord(c->ev_k0, s));
    nolsm_persist_kernel<<<c->p_grid, P_THREADS, P_SMEM_BYTES, s>>>(pe);
    CU_TRY(c, cudaGetLastError());
    CU_TRY(c, cudaEventRecord(c->ev_k1, s));
    c->t_launch = std::chrono::steady_clock::now();
    c->launch_seq += 1;
    c->launches = 1;
    c->rounds = 0;
    return NOLSM_OK;
}

}  // namespace

namespace nolsm_host {

int engine_create(nolsm_ctx* c) {
    c->eng = new (std::nothrow) Engine{};
    c->peng = new (std::nothrow) PEngine{};
    if (!c->eng || !c->peng) return fail(c, NOLSM_ENOMEM, "out of host memory");
    static_assert(P_MAX_MU == NOLSM_MAX_MU, "trial-mu capacity");
    if (use_umma(c)) CU_TRY(c, cudaFuncSetAttribute(nolsm_persist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SMEM_BYTES));
    return NOLSM_OK;
}

void engine_destroy(nolsm_ctx* c) {
    delete c->eng; c->eng = nullptr;
    delete c->peng; c->peng = nullptr;
}

int engine_block_keep(nolsm_ctx* c, unsigned char* d_keep, cudaStream_t s) {
    const int wpb = 8;
    const unsigned grid = (unsigned)((c->nnzb + wpb - 1) / wpb);
    if (c->val_dtype == NOLSM_DTYPE_F64)
        k_block_keep<double><<<grid, wpb * 32, 0, s>>>(c->d_blk_off, (const double*)c->dH, (const double*)c->dS, c->nnzb, c->opt.eps_filter, d_keep);
    else
        k_block_keep<float><<<grid, wpb * 32, 0, s>>>(c->d_blk_off, (const float*)c->dH, (const float*)c->dS, c->nnzb, c->opt.eps_filter, d_keep);
    CU_TRY(c, cudaGetLastError());
    return NOLSM_OK;
}

// Slots, workspace, tensor maps and the parameter blocks of both engines (the last part of nolsm_assemble).
int engine_plan(nolsm_ctx* c, cudaStream_t s) {
    int r;
    const int64_t n_atoms = c->n_atoms;
    Engine& e = *c->eng;
    e = Engine{};
    const size_t es = elem_size(c);
    const int max_n = c->max_n, max_nset = c->max_nset, max_nbi = c->max_nbi;
    double mean_tiles = 0, mean_n2 = 0;
    for (int64_t u = 0; u < c->n_units; ++u) {
        int ntm, ntn;
        choose_tiling((c->udim[u] + 15) & ~15, ntm, ntn);
        mean_tiles += (double)ntm * ntn;
        mean_n2 += (double)c->udim[u] * c->udim[u];
    }
    mean_tiles /= (double)c->n_units;
    mean_n2 /= (double)c->n_units;
    e.cap = (max_n + 15) & ~15;
    e.ld = (e.cap + 63) & ~63;                       // rows start on 128-byte lines: TMA boxes map to whole L2 lines
    e.bufsz = (long long)e.cap * e.ld;
    e.slotsz = e.bufsz * NBUF;
    size_t free_b = 0, total_b = 0;
    CU_TRY(c, cudaMemGetInfo(&free_b, &total_b));
    const size_t slot_bytes = (size_t)e.slotsz * es;
    const size_t cap_bytes = c->opt.workspace_bytes ? c->opt.workspace_bytes : std::min<size_t>(free_b / 2, (size_t)48 << 30);
    // persistent engine: the index tables and the dense strip of the gather task must fit the side group's shared memory
    c->persist = want_persist(c) && e.cap <= P_MAX_CAP && max_nbi <= NVC &&
                 (size_t)(3 * max_nset + 2) * 4 + (size_t)max_nset * 8 + 32 + G_STRIP_BYTES <= (size_t)P_SIDE_SMEM &&
                 (size_t)e.cap * 2 <= (size_t)G_STRIP_BYTES;
    if (c->combined && !c->persist) return fail(c, NOLSM_EINVAL, "combine: the groups do not fit the persistent engine (dimension or index-set size)");
    if (!c->persist && (c->opt.engine == NOLSM_ENGINE_PERSISTENT || c->opt.iteration == NOLSM_ITER_LOWDIN))
        return fail(c, NOLSM_EINVAL, "the persistent engine needs FP16/tcgen05 mode, submatrix dimensions <= 4096 and at most 16 basis functions per atom");
    // heavy-phase cap of the persistent engine: the live iterates of a slot in the GEMM chain are ~3.5 n^2 FP16
    // (X, T, next X / S, Y, R, next Y); the slots inside the chain together may fill L2 (heavy_slots sweep in profiles/r02_persist.md)
    int l2_bytes = 0;
    cudaDeviceGetAttribute(&l2_bytes, cudaDevAttrL2CacheSize, c->dev);
    if (l2_bytes <= 0) l2_bytes = 64 << 20;
    int g_max = (int)std::floor(1.0 * (double)l2_bytes / (3.5 * mean_n2 * 2.0));
    // the Loewdin form offers (ntm + 1) / 2 ntm of the tiles per GEMM (upper triangle only): twice as many chains keep the
    // CTA pairs busy (measured on cfg2: 24-28 against 12-14, profiles/r02_persist.md)
    if (c->opt.iteration == NOLSM_ITER_LOWDIN && c->opt.symmetric_tiles >= 0) g_max *= 2;
    g_max = std::max(3, std::min(g_max, 48));
    if (c->opt.heavy_slots > 0) g_max = c->opt.heavy_slots;
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
    int** res_i[] = {&e.at.inv, &e.at.sign, &e.at.status, &e.at.gemms, &c->d_gsym};
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
    if ((r = dmalloc(c, (void**)&c->d_mu_acc, 16 * NOLSM_MAX_MU))) return r;
    CU_TRY(c, cudaMemsetAsync(c->d_mu_acc, 0, 16 * NOLSM_MAX_MU, s));
    if (c->persist) {
        if (!encode_tiled_fn()) return fail(c, NOLSM_ECUDA, "cuTensorMapEncodeTiled not available");
        std::vector<CUtensorMap> maps((size_t)S * NMAP);
        const __half* vec0 = (const __half*)c->ws + (long long)S * e.slotsz;
        for (int sl = 0; sl < S; ++sl) {
            for (int b = 0; b < NBUF; ++b) {
                const __half* base = (const __half*)c->ws + (long long)sl * e.slotsz + (long long)b * e.bufsz;
                if (!make_tmap_f16_64x64(&maps[(size_t)sl * NMAP + b], base, e.cap, e.ld))
                    return fail(c, NOLSM_ECUDA, "cuTensorMapEncodeTiled failed");
            }
            for (int v = 0; v < 3; ++v) {       // the slot's two vector blocks, then the shared start block
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
    } else {
        r = c->opt.precision == NOLSM_PREC_FP32 ? set_smem_limits<float>(c) : set_smem_limits<__half>(c);
        if (r) return r;
    }
    if (c->persist) {
        PEngine& pe = *c->peng;
        pe = PEngine{};
        if ((r = dmalloc(c, (void**)&pe.slots, sizeof(PSlot) * S))) return r;
        if ((r = dmalloc(c, (void**)&pe.gclaim, 8 * S))) return r;
        if ((r = dmalloc(c, (void**)&pe.sclaim, 4 * S))) return r;
        if ((r = dmalloc(c, (void**)&pe.ctr, 8 * PC_LEN))) return r;
        if ((r = dmalloc(c, (void**)&c->d_abort, 4 * (1 + NOLSM_ABORT_HIST)))) return r;
        CU_TRY(c, cudaMemsetAsync(c->d_abort, 0, 4 * (1 + NOLSM_ABORT_HIST), s));
        c->launch_seq = c->checked_seq = 0;
        if ((r = dmalloc(c, (void**)&pe.heavy, 16))) return r;
        if ((r = dmalloc(c, (void**)&pe.pcols, (size_t)S * e.cap * PCW * sizeof(float)))) return r;
        if ((r = dmalloc(c, (void**)&pe.parked, 4 * S))) return r;
        pe.S = S; pe.cap = e.cap; pe.ld = e.ld; pe.bufsz = e.bufsz; pe.slotsz = e.slotsz;
        pe.tol_inv = e.tol_inv; pe.tol_sign = e.tol_sign; pe.max_inv = e.max_inv; pe.max_sign = e.max_sign;
        // Block power iteration (16 vectors, Frobenius growth): the estimate creeps up on rho from below (dense spectrum
        // edge: 0.75-0.80 rho after 3 steps, 0.84-0.87 after 6, 0.91-0.94 after 12 on the synthetic workloads), and an
        // overestimate is cheap (a factor 1.3 costs 0.3 scaled sign steps; the Schulz start converges for any
        // rho_hat > rho / 2) while an underestimate beyond 1.155 / alpha flips signs: few steps, generous safety, and for
        // rho(A) more steps (up to p_cap) while the estimate is visibly not settled (persist.cuh, p_tile_finished).
        pe.p_s = c->opt.power_iters_s > 0 ? c->opt.power_iters_s : 3;
        pe.p_a = c->opt.power_iters_a > 0 ? c->opt.power_iters_a : 6;
        pe.p_cap = std::max(pe.p_a, 24);
        pe.safety_s = pe.p_s >= 6 ? 1.05f : 1.3f;
        pe.safety_a = pe.p_a >= 12 ? 1.05f : pe.p_a >= 6 ? 1.25f : 1.45f;
        pe.gather_rowatoms = 4;
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
        pe.g_max = std::max(1, std::min(g_max, S));
        pe.want_lead = c->opt.tuning[0] > 0 ? c->opt.tuning[0] : G2_WANT_LEAD;
        pe.lowdin = c->opt.iteration == NOLSM_ITER_LOWDIN ? 1 : 0;
        pe.scan_rotate = c->opt.tuning[1] == 2 ? 1 : c->opt.tuning[1] == 1 ? 0 : (mean_n2 <= 768.0 * 768.0 ? 1 : 0);
        pe.l2_load = c->opt.tuning[2] > 0 ? c->opt.tuning[2] : 1; pe.l2_store = c->opt.tuning[3] > 0 ? c->opt.tuning[3] : 2;
        pe.sym_tiles = c->opt.symmetric_tiles >= 0 ? 1 : 0;
        pe.trans_tiles = c->opt.transposed_tiles >= 0 ? 1 : 0;
        pe.n_mu = 1; pe.count_only = 0;
        pe.nelec_mu = c->d_mu_acc; pe.e_mu = c->d_mu_acc + NOLSM_MAX_MU;
        pe.elem_chunks = 16;
        pe.dcols_chunks = 4;
        pe.next_atom = e.next_atom; pe.finished = e.finished; pe.abort_flag = c->d_abort;
        pe.at = e.at; pe.gsym = c->d_gsym; pe.sv = sys_view(c);
        pe.udim = c->d_udim; pe.upos = c->d_upos; pe.adim = c->d_dim;
        pe.S_vals = c->dS; pe.H_vals = c->dH; pe.val_f64 = c->val_dtype == NOLSM_DTYPE_F64;
        pe.e_atom = c->d_e_atom; pe.q_atom = c->d_q_atom; pe.maps = c->d_maps; pe.base = (__half*)c->ws;
        c->h_sclaim0.assign(S, ((unsigned)SK_REFILL << 28) | (1u << 14));
        {   // every CTA waits on work published by the others: the whole grid must be resident at once
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)(c->sms / 2 * 2)); cfg.blockDim = dim3(P_THREADS); cfg.dynamicSmemBytes = P_SMEM_BYTES;
            int ncl = 0;                      // the cluster shape (2, 1, 1) is a compile-time attribute of the kernel
            CU_TRY(c, cudaOccupancyMaxActiveClusters(&ncl, nolsm_persist_kernel, &cfg));
            if (ncl < 1) return fail(c, NOLSM_ECUDA, "no cluster of the persistent kernel fits on this device");
            c->p_grid = 2 * std::min(ncl, c->sms / 2);
        }
        CU_TRY(c, cudaFuncSetAttribute(k_side_gather<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SIDE_SMEM));
        CU_TRY(c, cudaFuncSetAttribute(k_side_gather<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SIDE_SMEM));
    }
    return NOLSM_OK;
}

int engine_run(nolsm_ctx* c, const double* mu, int n_mu, bool count_only, int64_t a0, int64_t a1, char* D_dev, int d_dtype, cudaStream_t) {
    c->ev_used = 0; c->recs.clear(); c->launches = 0; c->prof_on = false;
    c->last_persist = c->persist;
    c->n_mu_last = n_mu; c->last_count_only = count_only;
    if (c->persist) return run_persistent(c, mu, n_mu, count_only, a0, a1, D_dev, d_dtype);
    if (n_mu != 1 || count_only) return fail(c, NOLSM_EINVAL, "several trial mu per call need the persistent engine");
    return run_rounds(c, mu[0], a0, a1, D_dev, d_dtype);
}

int engine_status_bits(nolsm_ctx* c, int* bits) {
    const int64_t u0 = c->combined ? 0 : c->last_a0, nu = c->combined ? c->n_units : c->last_a1 - c->last_a0;   // status words are per unit
    std::vector<int> st(nu);
    CU_TRY(c, cudaMemcpy(st.data(), c->eng->at.status + u0, 4 * nu, cudaMemcpyDeviceToHost));
    int b = 0;
    if (c->combined) { for (int32_t u : c->h_feed) b |= st[u]; }           // the units of the last call
    else for (int64_t u = 0; u < nu; ++u) b |= st[u];
    *bits = b;
    return NOLSM_OK;
}

int engine_atom_stats(nolsm_ctx* c, int64_t a0, int64_t count, int32_t* dims, int32_t* inv_iters, int32_t* sign_iters,
                      int32_t* status, int32_t* gemms, float* residual, double* e_atom) {
    const Engine& e = *c->eng;
    if (c->combined) {
        // results are per unit: every member reports its unit's iteration counts, status and residual; the GEMMs and
        // the unit's dimension are reported by the unit's first member only (sums over atoms stay sums over units)
        const int64_t nu = c->n_units;
        std::vector<int32_t> ui(nu), us(nu), ut(nu), ug(nu), uy(nu);
        std::vector<float> ur(nu);
        CU_TRY(c, cudaMemcpy(ui.data(), e.at.inv, 4 * nu, cudaMemcpyDeviceToHost));
        CU_TRY(c, cudaMemcpy(us.data(), e.at.sign, 4 * nu, cudaMemcpyDeviceToHost));
        CU_TRY(c, cudaMemcpy(ut.data(), e.at.status, 4 * nu, cudaMemcpyDeviceToHost));
        CU_TRY(c, cudaMemcpy(ug.data(), e.at.gemms, 4 * nu, cudaMemcpyDeviceToHost));
        CU_TRY(c, cudaMemcpy(uy.data(), c->d_gsym, 4 * nu, cudaMemcpyDeviceToHost));
        CU_TRY(c, cudaMemcpy(ur.data(), e.at.res, 4 * nu, cudaMemcpyDeviceToHost));
        for (int64_t k = 0; k < count; ++k) {
            const int64_t a = a0 + k;
            const int32_t u = c->unit_of[a];
            const bool first = c->unit_mem[c->unit_ptr[u]] == a;
            if (dims) dims[k] = first ? c->udim[u] : 0;
            if (inv_iters) inv_iters[k] = ui[u];
            if (sign_iters) sign_iters[k] = us[u];
            if (status) status[k] = ut[u];
            if (gemms) gemms[k] = first ? ug[u] + uy[u] : 0;
            if (residual) residual[k] = ur[u];
        }
        if (e_atom) CU_TRY(c, cudaMemcpy(e_atom, c->d_e_atom + a0, 8 * count, cudaMemcpyDeviceToHost));
        return NOLSM_OK;
    }
    if (dims) memcpy(dims, c->dim.data() + a0, 4 * count);
    if (inv_iters) CU_TRY(c, cudaMemcpy(inv_iters, e.at.inv + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (sign_iters) CU_TRY(c, cudaMemcpy(sign_iters, e.at.sign + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (status) CU_TRY(c, cudaMemcpy(status, e.at.status + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (gemms) {
        std::vector<int32_t> gy(count);
        CU_TRY(c, cudaMemcpy(gemms, e.at.gemms + a0, 4 * count, cudaMemcpyDeviceToHost));
        CU_TRY(c, cudaMemcpy(gy.data(), c->d_gsym + a0, 4 * count, cudaMemcpyDeviceToHost));
        for (int64_t k = 0; k < count; ++k) gemms[k] += gy[k];
    }
    if (residual) CU_TRY(c, cudaMemcpy(residual, e.at.res + a0, 4 * count, cudaMemcpyDeviceToHost));
    if (e_atom) CU_TRY(c, cudaMemcpy(e_atom, c->d_e_atom + a0, 8 * count, cudaMemcpyDeviceToHost));
    return NOLSM_OK;
}

// FLOP one square GEMM of dimension n16 costs the tensor cores of the persistent pair engine, by the scheduler's tile rules
// (p_scheduler): 256 x bn tiles; symmetric products only on and above the diagonal; a ragged last row block transposed
// (M = 256 columns, N = the rows left) or, for its corner tile, as M = 128 when at most 128 rows are left.
static double padded_gemm_flops(int n16, bool sym, bool trans) {
    const int ntm = (n16 + BM - 1) / BM;
    double f = 0.0;
    for (int tm = 0; tm < ntm; ++tm)
        for (int tn = sym ? tm : 0; tn < ntm; ++tn) {
            const int bn = std::min(BN, n16 - tn * BN), rleft = n16 - tm * BM;
            if (trans && rleft < BM && tn < ntm - 1 && !sym) f += (double)BM * rleft;
            else if (rleft <= BM / 2 && (bn & 31) == 0) f += (double)(BM / 2) * bn;
            else f += (double)BM * bn;
        }
    return 2.0 * f * (double)n16;
}

// FLOP of the last call. A full GEMM counts 2 n^3. A symmetric product that multiplied only the tiles
// on and above the diagonal counts the share it executed, 2 n^3 (ntm + 1) / (2 ntm); flops_paper counts every GEMM at
// 2 n^3 (the paper's convention, which knows no symmetric products).
int engine_stats(nolsm_ctx* c, nolsm_stats* out) {
    const Engine& e = *c->eng;
    const int64_t nu = c->n_units;
    std::vector<int32_t> inv(nu), sg(nu), st(nu), gm(nu), gy(nu);
    CU_TRY(c, cudaMemcpy(inv.data(), e.at.inv, 4 * nu, cudaMemcpyDeviceToHost));
    CU_TRY(c, cudaMemcpy(sg.data(), e.at.sign, 4 * nu, cudaMemcpyDeviceToHost));
    CU_TRY(c, cudaMemcpy(st.data(), e.at.status, 4 * nu, cudaMemcpyDeviceToHost));
    CU_TRY(c, cudaMemcpy(gm.data(), e.at.gemms, 4 * nu, cudaMemcpyDeviceToHost));
    CU_TRY(c, cudaMemcpy(gy.data(), c->d_gsym, 4 * nu, cudaMemcpyDeviceToHost));
    std::vector<char> in_call(nu, 0);
    if (c->combined) for (int32_t u : c->h_feed) in_call[u] = 1;
    else for (int64_t u = c->last_a0; u < c->last_a1; ++u) in_call[u] = 1;
    for (int64_t u = 0; u < nu; ++u) {
        if (!in_call[u]) continue;
        out->sum_inv_iters += inv[u]; out->sum_sign_iters += sg[u];
        out->gemms_executed += gm[u] + gy[u];
        out->gemms_symmetric += gy[u];
        const double d = c->udim[u];
        const int n16 = (c->udim[u] + 15) & ~15;
        int ntm, ntn;
        choose_tiling(n16, ntm, ntn);
        const double fsym = (double)(ntm + 1) / (2.0 * ntm);
        out->flops_useful += 2.0 * d * d * d * (gm[u] + fsym * gy[u]);
        out->flops_paper += 2.0 * d * d * d * (gm[u] + gy[u]);
        // what the tensor cores executed: the persistent pair engine by its tile rules (padded_gemm_flops), the round
        // engine 256 rows per row block
        if (c->last_persist) {
            const bool sym = c->opt.symmetric_tiles >= 0, tr = c->opt.transposed_tiles >= 0;
            out->flops_padded += padded_gemm_flops(n16, false, tr) * gm[u] + padded_gemm_flops(n16, sym, tr) * gy[u];
        } else {
            out->flops_padded += 2.0 * (double)(ntm * BM) * (double)n16 * (double)n16 * (gm[u] + gy[u]);
        }
        out->n_notspd += (st[u] & ST_NOTSPD) ? 1 : 0;
        out->n_noconv += (st[u] & ST_NOCONV) ? 1 : 0;
        out->gather_bytes += 2.0 * (double)n16 * (double)n16 * elem_size(c);      // dense S_sub and H_sub written (once per unit)
    }
    const size_t es = elem_size(c), vs = c->val_dtype == NOLSM_DTYPE_F64 ? 8 : 4;
    for (int64_t i = c->last_a0; i < c->last_a1; ++i) {
        const double n = c->dim[i];
        const double nv = (double)(c->blk_off[c->row_ptr[i + 1]] - c->blk_off[c->row_ptr[i]]);
        out->scatter_bytes += nv * (c->last_ds + vs) + (n * n + n * c->atom_nb[i]) * es;
    }
    return NOLSM_OK;
}

int engine_profile(nolsm_ctx* c, double* out) {
    if (c->last_persist) {
        // one launch: the kernel's duration from CUDA events on its stream; side-task times are summed
        // over the side groups (SM-time, the tasks run concurrently with the GEMM pipeline)
        unsigned long long ct[PC_LEN];
        CU_TRY(c, cudaMemcpy(ct, c->peng->ctr, sizeof(ct), cudaMemcpyDeviceToHost));
        float kms = 0;
        CU_TRY(c, cudaEventElapsedTime(&kms, c->ev_k0, c->ev_k1));
        nolsm_stats st;
        if (int r = nolsm_get_stats(c, &st)) return r;
        out[0] = ct[PC_SIDE_NS + SK_GATHER] * 1e-6; out[1] = (double)ct[PC_SIDE_TASKS + SK_GATHER]; out[2] = (double)ct[PC_SIDE_BYTES + SK_GATHER];
        out[3] = kms; out[4] = 1; out[5] = st.flops_useful; out[6] = st.flops_padded;
        out[7] = ct[PC_SIDE_NS + SK_DCOLS] * 1e-6; out[8] = (double)ct[PC_SIDE_TASKS + SK_DCOLS]; out[9] = (double)ct[PC_SIDE_BYTES + SK_DCOLS];
        out[10] = (ct[PC_SIDE_NS + SK_REFILL] + ct[PC_SIDE_NS + SK_ELEM] + ct[PC_SIDE_NS + SK_WCOLS]) * 1e-6;
        out[11] = (double)(ct[PC_SIDE_TASKS + SK_REFILL] + ct[PC_SIDE_TASKS + SK_ELEM] + ct[PC_SIDE_TASKS + SK_WCOLS]);
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
    CU_TRY(c, cudaMemcpy(pf, c->eng->prof, sizeof(pf), cudaMemcpyDeviceToHost));
    const size_t es = elem_size(c), vs = c->val_dtype == NOLSM_DTYPE_F64 ? 8 : 4;
    out[0] = ms[K_GATHER]; out[1] = cnt[K_GATHER]; out[2] = pf[PF_GATHER_SRC] * vs + pf[PF_GATHER_DENSE] * es;
    out[3] = ms[K_GEMM]; out[4] = cnt[K_GEMM]; out[5] = pf[PF_FLOP_USEFUL]; out[6] = pf[PF_FLOP_PADDED];
    out[7] = ms[K_DCOLS]; out[8] = cnt[K_DCOLS]; out[9] = pf[PF_DCOLS_BYTES];
    out[10] = ms[K_OTHER]; out[11] = cnt[K_OTHER];
    out[12] = pf[PF_SUBMATS]; out[13] = (double)c->launches;
    return NOLSM_OK;
}

int engine_counters(nolsm_ctx* c, double* out) {
    for (int i = 0; i < NOLSM_COUNTERS_LEN; ++i) out[i] = 0;
    if (!c->last_persist) return NOLSM_OK;
    unsigned long long ct[PC_LEN];
    CU_TRY(c, cudaMemcpy(ct, c->peng->ctr, sizeof(ct), cudaMemcpyDeviceToHost));
    float kms = 0;
    CU_TRY(c, cudaEventElapsedTime(&kms, c->ev_k0, c->ev_k1));
    out[0] = 1; out[1] = kms; out[2] = (double)(ct[PC_T_END] - ct[PC_T_START]) * 1e-6;
    out[3] = (double)ct[PC_TILES]; out[4] = ct[PC_SCHED_IDLE_NS] * 1e-6; out[5] = ct[PC_SCHED_BUSY_NS] * 1e-6;
    out[6] = (double)ct[PC_OVERSHOOT]; out[7] = c->peng->S; out[8] = c->p_grid / 2;
    for (int k = 0; k < 8; ++k) {
        out[9 + k] = ct[PC_SIDE_NS + k] * 1e-6;
        out[17 + k] = (double)ct[PC_SIDE_BYTES + k];
        out[25 + k] = (double)ct[PC_SIDE_TASKS + k];
    }
    for (int k = 0; k < 3; ++k) out[33 + k] = ct[PC_MMA_NS + k] * 1e-6;
    out[36] = ct[PC_SCHED_RING_NS] * 1e-6; out[37] = ct[PC_SCHED_CREDIT_NS] * 1e-6;
    out[38] = (double)ct[PC_POW_EXTRA];
    return NOLSM_OK;
}

// The gather kernel for one atom's submatrix (is_unit: one unit's union submatrix), copied to the host tight.
int engine_gather(nolsm_ctx* c, int64_t id, bool is_unit, int which, int out_fp16, void* out_host) {
    const size_t es = out_fp16 ? 2 : 4;
    const Engine& e0 = *c->eng;
    if ((size_t)e0.slotsz * es > c->ws_bytes) return fail(c, NOLSM_ENOMEM, "workspace too small for an FP32 gather");
    if (c->persist && out_fp16) {
        // the gather task of the persistent engine, launched stand-alone into slot 0
        const int64_t unit = is_unit ? id : (c->combined ? -1 : id);
        if (unit < 0) return fail(c, NOLSM_ESTATE, "with combine the dense submatrices are per group: nolsm_gather_submatrix maps the atom to its unit");
        DevBuf unit_buf;
        CU_TRY(c, cudaMalloc(&unit_buf.p, 4));
        int* d_unit = unit_buf.as<int>();
        const int u32 = (int)unit;
        CU_TRY(c, cudaMemcpy(d_unit, &u32, 4, cudaMemcpyHostToDevice));
        const PEngine& pe = *c->peng;
        const int nset = (int)(c->uset_ptr[unit + 1] - c->uset_ptr[unit]);
        dim3 grid((nset + pe.gather_rowatoms - 1) / pe.gather_rowatoms, 1);
        if (c->val_dtype == NOLSM_DTYPE_F64)
            k_side_gather<double><<<grid, P_SIDE_THREADS, P_SIDE_SMEM, c->s_main>>>(pe.sv, (const double*)c->dS, (const double*)c->dH, pe.base, pe.slotsz, pe.bufsz, pe.ld, d_unit, c->d_udim, 1, nullptr);
        else
            k_side_gather<float><<<grid, P_SIDE_THREADS, P_SIDE_SMEM, c->s_main>>>(pe.sv, (const float*)c->dS, (const float*)c->dH, pe.base, pe.slotsz, pe.bufsz, pe.ld, d_unit, c->d_udim, 1, nullptr);
        cudaError_t ce = cudaGetLastError();
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(c->s_main);
        const int n = c->udim[unit];
        if (ce == cudaSuccess)
            ce = cudaMemcpy2D(out_host, (size_t)n * 2, (const char*)c->ws + (size_t)which * pe.bufsz * 2, (size_t)pe.ld * 2,
                              (size_t)n * 2, n, cudaMemcpyDeviceToHost);
        if (ce != cudaSuccess) { c->err = cudaGetErrorString(ce); return NOLSM_ECUDA; }
        return NOLSM_OK;
    }
    if (is_unit || c->combined) return fail(c, NOLSM_ESTATE, "unit gathers need the persistent engine and FP16 output");
    // a one-slot view of the round engine with the slot forced into phase NEW
    const int64_t atom = id;
    Engine e = e0;
    e.S = 1;
    e.profiling = 0;
    Slot sl{};
    sl.atom = (int)atom; sl.n = c->dim[atom]; sl.n16 = (sl.n + 15) & ~15; sl.pos = c->pos[atom]; sl.nbi = c->atom_nb[atom];
    sl.phase = sl.snap = PH_NEW;
    DevBuf slot_buf;
    CU_TRY(c, cudaMalloc(&slot_buf.p, sizeof(Slot)));
    Slot* d_sl = slot_buf.as<Slot>();
    CU_TRY(c, cudaMemcpy(d_sl, &sl, sizeof(Slot), cudaMemcpyHostToDevice));
    e.slots = d_sl;
    int r;
    if (out_fp16) { r = set_smem_limits<__half>(c); if (!r) r = launch_gather<__half>(c, e, c->max_nset, c->s_main); }
    else { r = set_smem_limits<float>(c); if (!r) r = launch_gather<float>(c, e, c->max_nset, c->s_main); }
    if (!r) {
        cudaError_t ce = cudaStreamSynchronize(c->s_main);
        if (ce == cudaSuccess)
            ce = cudaMemcpy2D(out_host, (size_t)sl.n * es, (const char*)c->ws + (size_t)which * e.bufsz * es,
                              (size_t)e.ld * es, (size_t)sl.n * es, sl.n, cudaMemcpyDeviceToHost);
        if (ce != cudaSuccess) { c->err = cudaGetErrorString(ce); r = NOLSM_ECUDA; }
    }
    return r;
}

// Stand-alone timing of the two HBM-bound side tasks: which = 0 the gather of every unit (a1), 1 the D
// columns + scatter + energy of every atom (a6-a7; the slot operands hold whatever the last call left, the arithmetic is
// the same). The same device functions as inside the persistent kernel, one side group per CTA, a full wave of CTAs;
// `reps` launches, CUDA events around them. bytes_out = algorithmic bytes of one launch.
int engine_side_bandwidth(nolsm_ctx* c, int which, int reps, double* ms_out, double* bytes_out) {
    if (!c->persist) return fail(c, NOLSM_ESTATE, "side-task bandwidth needs the persistent engine");
    if (which == 1 && c->combined) return fail(c, NOLSM_ESTATE, "scatter bandwidth: assemble without combine");
    const PEngine& pe = *c->peng;
    cudaStream_t s = c->s_main;
    EventPair evp;
    CU_TRY(c, cudaEventCreate(&evp.a));
    CU_TRY(c, cudaEventCreate(&evp.b));
    const cudaEvent_t e0 = evp.a, e1 = evp.b;
    const int64_t count = which == 0 ? c->n_units : c->n_atoms;
    std::vector<int> ids(count);
    for (int64_t i = 0; i < count; ++i) ids[i] = (int)i;
    DevBuf ids_buf, bytes_buf;
    CU_TRY(c, cudaMalloc(&ids_buf.p, 4 * count));
    int* d_ids = ids_buf.as<int>();
    CU_TRY(c, cudaMemcpy(d_ids, ids.data(), 4 * count, cudaMemcpyHostToDevice));
    CU_TRY(c, cudaMalloc(&bytes_buf.p, 8));
    unsigned long long* d_bytes = bytes_buf.as<unsigned long long>();
    CU_TRY(c, cudaMemset(d_bytes, 0, 8));
    double bytes = 0;
    const size_t vs = c->val_dtype == NOLSM_DTYPE_F64 ? 8 : 4;
    const int64_t per_launch = 65535;                 // gridDim.y limit
    auto launch_all = [&](bool count_bytes) -> cudaError_t {
        for (int64_t b = 0; b < count; b += per_launch) {
            const int m = (int)std::min<int64_t>(per_launch, count - b);
            if (which == 0) {
                const int chunks = (c->max_nset + pe.gather_rowatoms - 1) / pe.gather_rowatoms;
                dim3 grid(chunks, m);
                if (c->val_dtype == NOLSM_DTYPE_F64)
                    k_side_gather<double><<<grid, P_SIDE_THREADS, P_SIDE_SMEM, s>>>(pe.sv, (const double*)c->dS, (const double*)c->dH, pe.base, pe.slotsz, pe.bufsz, pe.ld, d_ids + b, c->d_udim, pe.S, count_bytes ? d_bytes : nullptr);
                else
                    k_side_gather<float><<<grid, P_SIDE_THREADS, P_SIDE_SMEM, s>>>(pe.sv, (const float*)c->dS, (const float*)c->dH, pe.base, pe.slotsz, pe.bufsz, pe.ld, d_ids + b, c->d_udim, pe.S, count_bytes ? d_bytes : nullptr);
            } else {
                dim3 grid(pe.dcols_chunks, m);
                const size_t smem = (size_t)(2 * c->max_nset + 2) * 4;
                double* Dd = (double*)c->d_D_stage;
                if (c->val_dtype == NOLSM_DTYPE_F64)
                    k_side_dcols<double, double><<<grid, P_SIDE_THREADS, smem, s>>>(pe.sv, pe.pcols, pe.base, pe.slotsz, 2 * pe.bufsz, pe.cap, pe.ld, d_ids + b, c->d_dim, c->d_upos, c->d_atom_nb, pe.S, (const double*)c->dH, (const double*)c->dS, Dd, c->d_e_atom, c->d_q_atom);
                else
                    k_side_dcols<float, double><<<grid, P_SIDE_THREADS, smem, s>>>(pe.sv, pe.pcols, pe.base, pe.slotsz, 2 * pe.bufsz, pe.cap, pe.ld, d_ids + b, c->d_dim, c->d_upos, c->d_atom_nb, pe.S, (const float*)c->dH, (const float*)c->dS, Dd, c->d_e_atom, c->d_q_atom);
            }
        }
        return cudaGetLastError();
    };
    if (which == 1) {
        const size_t need = (size_t)c->nvals * 8;
        if (c->d_D_stage_bytes < need) {
            if (c->d_D_stage) cudaFree(c->d_D_stage);
            c->d_D_stage = nullptr; c->d_D_stage_bytes = 0;
            CU_TRY(c, cudaMalloc(&c->d_D_stage, need));
            c->d_D_stage_bytes = need;
        }
        for (int64_t i = 0; i < c->n_atoms; ++i) {
            const double nv = (double)(c->blk_off[c->row_ptr[i + 1]] - c->blk_off[c->row_ptr[i]]);
            bytes += nv * (8 + 2 * vs) + (double)c->dim[i] * PCW * 4.0 + (double)c->dim[i] * c->atom_nb[i] * 2.0;
        }
    }
    CU_TRY(c, launch_all(which == 0));                // warm-up; the gather counts its own bytes once
    CU_TRY(c, cudaStreamSynchronize(s));
    if (which == 0) {
        unsigned long long hb = 0;
        CU_TRY(c, cudaMemcpy(&hb, d_bytes, 8, cudaMemcpyDeviceToHost));
        bytes = (double)hb;
    }
    CU_TRY(c, cudaEventRecord(e0, s));
    for (int r = 0; r < reps; ++r) CU_TRY(c, launch_all(false));
    CU_TRY(c, cudaEventRecord(e1, s));
    CU_TRY(c, cudaEventSynchronize(e1));
    float ms = 0;
    CU_TRY(c, cudaEventElapsedTime(&ms, e0, e1));
    *ms_out = ms / reps;
    *bytes_out = bytes;
    c->have_result = false;                           // the energies of the last call were overwritten
    return NOLSM_OK;
}

}  // namespace nolsm_host

// =====================================================================================================================
// nolsm_gather_submatrix_noalloc (include/nolsm.h): the gather task a1 for one submatrix without any device allocation.
//
// For callers that cannot allocate: all device memory already belongs to the host program's own pool, or a cudaMalloc /
// cudaFree (which wait for the whole device) would stall behind kernels that are still running. The dense, padded
// T(S) | T(H0) pair that the existing path puts into workspace slot 0 goes into the array below instead, which is part of
// the library image: 2 * 2048^2 FP16 values = 16 MiB on every GPU that loads this library, until the process exits.
//
// The name `g_noalloc_scratch` is a device address only inside device code. In host code it names a host-side shadow
// object; handing that to a kernel makes the kernel fault (or, on systems where the GPU can reach host memory, scribble
// over the shadow). Host code therefore asks the runtime for the device address, once per device with that device
// current (noalloc_setup), and passes the returned pointer to the kernel.
// =====================================================================================================================
#include <mutex>

constexpr int NOALLOC_MAX_DIM = NOLSM_NOALLOC_MAX_DIM;
constexpr size_t NOALLOC_HALVES = 2ull * NOALLOC_MAX_DIM * NOALLOC_MAX_DIM;
static_assert(NOALLOC_MAX_DIM % 16 == 0, "rows of the scratch matrices are written with 16-byte stores");
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_HALVES * sizeof(__half)];

namespace nolsm {
// side_gather_chunk of the persistent kernel (persist.cuh) launched alone like k_side_gather, but the unit and its
// dimension come by value (no device-side id list) and the two dense matrices go to `scratch` | `scratch + bufsz`.
// grid = chunks of row-atoms, one 128-thread side group per CTA.
template <typename TV>
__global__ void __launch_bounds__(P_SIDE_THREADS) k_side_gather_scratch(SysView sv, const TV* S_vals, const TV* H_vals, __half* scratch,
                                                                        long long bufsz, int ld, int unit, int n) {
    extern __shared__ unsigned char sm_dyn[];
    side_gather_chunk<TV>(sv, S_vals, H_vals, scratch, scratch + bufsz, unit, n, (n + 15) & ~15, ld, blockIdx.x, gridDim.x, sm_dyn,
                          threadIdx.x, nullptr);
}
}  // namespace nolsm

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
__half* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};      // device address of g_noalloc_scratch on device d, once looked up

// Once per device and process, with that device current: the device address of the scratch array and the shared-memory
// limit of the two kernel instances. Neither call allocates device memory.
int noalloc_setup(nolsm_ctx* c, __half** out) {
    int dev = -1;
    CU_TRY(c, cudaGetDevice(&dev));
    if (dev != c->dev) { CU_TRY(c, cudaSetDevice(c->dev)); dev = c->dev; }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(c, NOLSM_EINVAL, "nolsm_gather_submatrix_noalloc: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void* p = nullptr;
        CU_TRY(c, cudaGetSymbolAddress(&p, g_noalloc_scratch));
        CU_TRY(c, cudaFuncSetAttribute(k_side_gather_scratch<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SIDE_SMEM));
        CU_TRY(c, cudaFuncSetAttribute(k_side_gather_scratch<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SIDE_SMEM));
        g_noalloc_ptr[dev] = static_cast<__half*>(p);
    }
    *out = g_noalloc_ptr[dev];
    return NOLSM_OK;
}
}  // namespace

namespace nolsm_host {

// Gathers unit `unit` (an atom without combination) into the static scratch array and copies matrix `which` tight to
// `out` (device: asynchronous on s; host: the call waits). No cudaMalloc / cudaFree / allocating routine on this path.
// Every element the copy reads is written by the kernel of the same call (zero-filled strips, then the blocks), so the
// contents the previous call left behind need no clearing. Calls that overlap on the GPU race on the array.
int engine_gather_noalloc(nolsm_ctx* c, int64_t unit, int which, void* out, cudaStream_t s) {
    if (!c->persist) return fail(c, NOLSM_ESTATE, "nolsm_gather_submatrix_noalloc needs the persistent engine (FP16 operands)");
    const int n = c->udim[unit], n16 = (n + 15) & ~15;
    if (n16 > NOALLOC_MAX_DIM)
        return fail(c, NOLSM_EINVAL, "nolsm_gather_submatrix_noalloc: padded submatrix dimension " + std::to_string(n16) +
                                         " exceeds NOLSM_NOALLOC_MAX_DIM = " + std::to_string(NOALLOC_MAX_DIM) +
                                         " (the static scratch array holds two 2048 x 2048 FP16 matrices); use nolsm_gather_submatrix");
    __half* scratch = nullptr;
    if (int r = noalloc_setup(c, &scratch)) return r;
    const PEngine& pe = *c->peng;
    const int nset = (int)(c->uset_ptr[unit + 1] - c->uset_ptr[unit]);
    const long long bufsz = (long long)n16 * n16;
    const int ld = n16;
    const dim3 grid((nset + pe.gather_rowatoms - 1) / pe.gather_rowatoms, 1);
    if (c->val_dtype == NOLSM_DTYPE_F64)
        k_side_gather_scratch<double><<<grid, P_SIDE_THREADS, P_SIDE_SMEM, s>>>(pe.sv, (const double*)c->dS, (const double*)c->dH, scratch,
                                                                                 bufsz, ld, (int)unit, n);
    else
        k_side_gather_scratch<float><<<grid, P_SIDE_THREADS, P_SIDE_SMEM, s>>>(pe.sv, (const float*)c->dS, (const float*)c->dH, scratch,
                                                                                bufsz, ld, (int)unit, n);
    CU_TRY(c, cudaGetLastError());
    const bool on_device = is_device_ptr(out);
    CU_TRY(c, cudaMemcpy2DAsync(out, (size_t)n * 2, scratch + (size_t)which * bufsz, (size_t)ld * 2, (size_t)n * 2, n,
                                on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s));
    if (!on_device) CU_TRY(c, cudaStreamSynchronize(s));
    return NOLSM_OK;
}

}  // namespace nolsm_host
