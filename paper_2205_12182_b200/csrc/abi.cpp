// C ABI of the NOLSM hot path (include/nolsm.h): context life cycle, the density-matrix calls, results and
// diagnostics. Host code only; every step of the path runs in the kernels behind engine.cu.
#include <cmath>

#include "ctx.h"

using namespace nolsm_host;

namespace nolsm_host {

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
void free_assembled(nolsm_ctx* c, bool release) {
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

// The abort words of every persistent launch since the last check: the running word of the last launch and the saved
// final words of the launches before it (run_persistent saves a launch's word before the next launch clears it, so a
// stalled kernel in a series of nolsm_density_matrix_range calls is not forgotten). Call after the stream has drained.
int check_abort_words(nolsm_ctx* c) {
    if (c->launch_seq == c->checked_seq) return NOLSM_OK;
    int w[1 + NOLSM_ABORT_HIST] = {};
    CU_TRY(c, cudaMemcpy(w, c->d_abort, sizeof(w), cudaMemcpyDeviceToHost));
    int worst = w[0];
    int64_t first_bad = w[0] ? c->launch_seq - 1 : -1;
    for (int64_t k = c->launch_seq - 2; k >= c->checked_seq; --k)
        if (w[1 + k % NOLSM_ABORT_HIST]) { worst = std::max(worst, w[1 + k % NOLSM_ABORT_HIST]); first_bad = k; }
    const int64_t n_calls = c->launch_seq - c->checked_seq;
    c->checked_seq = c->launch_seq;
    if (!worst) return NOLSM_OK;
    c->have_result = false;
    const std::string which = n_calls > 1 ? " (call " + std::to_string(first_bad - (c->launch_seq - n_calls) + 1) + " of the " +
                                                std::to_string(n_calls) + " since the last wait; rows written since then are incomplete)" : "";
    c->err = (worst == 2 ? "persistent engine: a wait inside the kernel stalled (device watchdog); the results of this call are invalid"
                         : "persistent engine exceeded its time limit and was aborted") + which;
    return NOLSM_ECUDA;
}

// Waits for the last density_matrix call. The persistent kernel is watched: past the time limit (counted from its
// launch) the host raises the kernel's abort word (copy on a second stream), which makes the tile schedulers stop
// feeding and every role leave its loop. A wait inside the kernel that stalls raises the same word itself (value 2,
// gemm_umma.cuh). A pageable host D is copied here, after the watched wait, so the watchdog also covers that case.
int wait_result(nolsm_ctx* c) {
    if (c->last_persist) {
        bool aborted = false;
        for (;;) {
            const cudaError_t q = cudaEventQuery(c->ev_out);
            if (q == cudaSuccess) break;
            if (q != cudaErrorNotReady) { c->err = std::string("persistent engine: ") + cudaGetErrorString(q); return NOLSM_ECUDA; }
            const double el = std::chrono::duration<double>(std::chrono::steady_clock::now() - c->t_launch).count();
            if (!aborted && el > c->timeout_s) {
                static const int one = 1;
                cudaMemcpyAsync(c->d_abort, &one, 4, cudaMemcpyHostToDevice, c->s_x);
                aborted = true;
            }
            if (el > c->timeout_s + 60.0) { c->err = "persistent engine did not stop after abort"; return NOLSM_ECUDA; }
            std::this_thread::sleep_for(std::chrono::microseconds(el < 0.01 ? 20 : 200));
        }
        if (int r = check_abort_words(c)) { c->pend_dst = nullptr; return r; }
    }
    CU_TRY(c, cudaStreamSynchronize(c->last_stream));
    if (c->pend_dst) {
        void* dst = c->pend_dst;
        c->pend_dst = nullptr;
        CU_TRY(c, cudaMemcpy(dst, c->d_D_stage, c->pend_bytes, cudaMemcpyDeviceToHost));
    }
    return NOLSM_OK;
}

}  // namespace nolsm_host

namespace {

// Common front end of the calls that run the engine: output staging, stream ordering, zeroing of the outputs.
int run(nolsm_ctx* c, const double* mu, int n_mu, bool count_only, int64_t a0, int64_t a1, void* D_vals, int d_dtype, void* cuda_stream) {
    cudaStream_t us = (cudaStream_t)cuda_stream;
    cudaStream_t s = c->s_main;
    cudaSetDevice(c->dev);
    if (c->pend_dst) { if (int r = wait_result(c)) return r; }      // the staged D of the previous call goes home first
    const size_t ds = d_dtype == NOLSM_DTYPE_F64 ? 8 : 4;
    c->last_ds = ds;
    const int64_t v0 = c->blk_off[c->row_ptr[a0]], v1 = c->blk_off[c->row_ptr[a1]];
    // device view of the output rows [a0, a1): D_dev points at element 0 of the whole array
    char* D_dev = nullptr;
    const bool host_out = !count_only && !is_device_ptr(D_vals);
    if (host_out) {
        const size_t need = (size_t)(v1 - v0) * ds;
        if (c->d_D_stage_bytes < need) {
            if (c->d_D_stage) cudaFree(c->d_D_stage);
            c->d_D_stage = nullptr; c->d_D_stage_bytes = 0;
            CU_TRY(c, cudaMalloc(&c->d_D_stage, need));
            c->d_D_stage_bytes = need;
        }
        D_dev = (char*)c->d_D_stage - (size_t)v0 * ds;
    } else if (!count_only) {
        D_dev = (char*)D_vals;
    }
    // the engine runs on the library's own stream; it is ordered after the caller's stream and the caller's stream
    // after it
    CU_TRY(c, cudaEventRecord(c->ev_in, us));
    CU_TRY(c, cudaStreamWaitEvent(s, c->ev_in, 0));
    if (!count_only) CU_TRY(c, cudaMemsetAsync(D_dev + (size_t)v0 * ds, 0, (size_t)(v1 - v0) * ds, s));
    CU_TRY(c, cudaMemsetAsync(c->d_e_atom + a0, 0, 8 * (a1 - a0), s));
    CU_TRY(c, cudaMemsetAsync(c->d_q_atom + a0, 0, 8 * (a1 - a0), s));
    if (int r = engine_run(c, mu, n_mu, count_only, a0, a1, D_dev, d_dtype, s)) return r;
    if (host_out) {
        // pinned memory: the copy is enqueued behind the kernel and the call returns. Pageable memory: the copy would block
        // this thread until the kernel has ended, with nobody watching the time limit; wait_result does it instead.
        cudaPointerAttributes at{};
        const bool pinned = cudaPointerGetAttributes(&at, D_vals) == cudaSuccess && at.type == cudaMemoryTypeHost;
        cudaGetLastError();
        if (pinned) CU_TRY(c, cudaMemcpyAsync((char*)D_vals + (size_t)v0 * ds, c->d_D_stage, (size_t)(v1 - v0) * ds, cudaMemcpyDeviceToHost, s));
        else { c->pend_dst = (char*)D_vals + (size_t)v0 * ds; c->pend_bytes = (size_t)(v1 - v0) * ds; }
    }
    CU_TRY(c, cudaEventRecord(c->ev_out, s));
    CU_TRY(c, cudaStreamWaitEvent(us, c->ev_out, 0));
    c->last_stream = us; c->last_a0 = a0; c->last_a1 = a1; c->have_result = true;
    return NOLSM_OK;
}

}  // namespace

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

int nolsm_abi_version(void) { return NOLSM_ABI_VERSION; }
size_t nolsm_sizeof_options(void) { return sizeof(nolsm_options); }
size_t nolsm_sizeof_stats(void) { return sizeof(nolsm_stats); }

int nolsm_create(nolsm_ctx** out, int cuda_device, const nolsm_options* opt) try {
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
    bool bad = o.precision != NOLSM_PREC_FP16_FP32 && !fp32;
    if (o.max_inv_iters <= 0) o.max_inv_iters = 24;
    if (o.max_sign_iters <= 0) o.max_sign_iters = 64;
    if (o.tol_inv <= 0) o.tol_inv = fp32 ? 1e-5f : 2e-3f;
    if (o.tol_sign <= 0) o.tol_sign = fp32 ? 1e-5f : 2e-3f;
    if (o.power_iters_s < 0) o.power_iters_s = 0;      // 0 = default of the engine that runs (assemble)
    if (o.power_iters_a < 0) o.power_iters_a = 0;
    bad = bad || o.eps_filter < 0;
    if (o.sign_scaled_iters == 0) o.sign_scaled_iters = 6;
    if (o.sign_scaled_iters < 0) o.sign_scaled_iters = 0;
    if (o.sign_scaled_iters > 14) o.sign_scaled_iters = 14;
    bad = bad || o.combine < 0 || o.combine > 2;
    if (o.combine_max_dim <= 0) o.combine_max_dim = 2048;
    if (o.combine_max_members <= 0) o.combine_max_members = 16;
    if (o.combine_max_candidates <= 0) o.combine_max_candidates = 24;
    if (o.sign_scale == 0.f) o.sign_scale = 1.5f;
    bad = bad || !(o.sign_scale > 1.f && o.sign_scale < 1.7320508f);
    bad = bad || o.engine < 0 || o.engine > NOLSM_ENGINE_ROUNDS;
    bad = bad || o.iteration < 0 || o.iteration > NOLSM_ITER_LOWDIN;
    bad = bad || o.heavy_slots < 0 || o.tuning[0] < 0;
    if (bad) { delete c; return NOLSM_EINVAL; }
    cudaSetDevice(cuda_device);
    cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, cuda_device);
    if (o.timeout_s > 0) c->timeout_s = o.timeout_s;
    bool ok = cudaStreamCreateWithFlags(&c->s_main, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&c->s_x, cudaStreamNonBlocking) == cudaSuccess;
    cudaEvent_t* evs[] = {&c->ev_in, &c->ev_out};
    for (cudaEvent_t* e : evs) ok = ok && cudaEventCreateWithFlags(e, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < NOLSM_ROUND_DEPTH; ++i) ok = ok && cudaEventCreateWithFlags(&c->ev_round[i], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaEventCreate(&c->ev_k0) == cudaSuccess && cudaEventCreate(&c->ev_k1) == cudaSuccess;
    ok = ok && engine_create(c) == NOLSM_OK;
    if (!ok) { cudaGetLastError(); nolsm_destroy(c); return NOLSM_ECUDA; }   // releases the streams and events that exist
    *out = c;
    return NOLSM_OK;
} catch (...) { return NOLSM_ENOMEM; }

int nolsm_destroy(nolsm_ctx* c) try {
    if (!c) return NOLSM_EINVAL;
    cudaSetDevice(c->dev);
    free_assembled(c, true);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    cudaEvent_t evs[] = {c->ev_in, c->ev_out, c->ev_k0, c->ev_k1};
    for (cudaEvent_t e : evs) if (e) cudaEventDestroy(e);
    for (int i = 0; i < NOLSM_ROUND_DEPTH; ++i) if (c->ev_round[i]) cudaEventDestroy(c->ev_round[i]);
    if (c->s_main) cudaStreamDestroy(c->s_main);
    if (c->s_x) cudaStreamDestroy(c->s_x);
    engine_destroy(c);
    delete c;
    return NOLSM_OK;
} catch (...) { return on_exception(c, "nolsm_destroy"); }

const char* nolsm_last_error(const nolsm_ctx* c) { return c ? c->err.c_str() : "null context"; }

int nolsm_set_perf_table(nolsm_ctx* c, const int32_t* n, const double* tflops, int count) try {
    if (!c) return NOLSM_EINVAL;
    if (count == 0) { c->pn_n.clear(); c->pn_rate.clear(); return NOLSM_OK; }
    if (!n || !tflops || count < 0) return fail(c, NOLSM_EINVAL, "null table");
    std::vector<int64_t> tn(count), tr(count);
    for (int k = 0; k < count; ++k) {
        tn[k] = n[k];
        tr[k] = (int64_t)std::llround(tflops[k] * 1000.0);            // GFLOP/s, integer
        if (tn[k] <= 0 || tn[k] > 8192 || tr[k] <= 0 || (k > 0 && tn[k] <= tn[k - 1]))
            return fail(c, NOLSM_EINVAL, "perf table: dimensions must ascend strictly within 1..8192, rates must be positive");
    }
    c->pn_n = tn; c->pn_rate = tr;
    return NOLSM_OK;
} catch (...) { return on_exception(c, "nolsm_set_perf_table"); }

int nolsm_density_matrix_range(nolsm_ctx* c, double mu, int64_t a0, int64_t a1, void* D_vals, int d_dtype,
                               double* e_partial_host, void* cuda_stream) try {
    if (!c) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "nolsm_assemble has not been called");
    if (!D_vals || a0 < 0 || a1 > c->n_atoms || a0 >= a1) return fail(c, NOLSM_EINVAL, "bad range or null D_vals");
    if (d_dtype != NOLSM_DTYPE_F64 && d_dtype != NOLSM_DTYPE_F32) return fail(c, NOLSM_EINVAL, "bad d_dtype");
    if (int r = run(c, &mu, 1, false, a0, a1, D_vals, d_dtype, cuda_stream)) return r;
    if (e_partial_host) return nolsm_energy(c, e_partial_host);
    return NOLSM_OK;
} catch (...) { return on_exception(c, "nolsm_density_matrix_range"); }

int nolsm_density_matrix(nolsm_ctx* c, double mu, void* D_vals, int d_dtype, void* cuda_stream) try {
    if (!c) return NOLSM_EINVAL;
    return nolsm_density_matrix_range(c, mu, 0, c->n_atoms, D_vals, d_dtype, nullptr, cuda_stream);
} catch (...) { return on_exception(c, "nolsm_density_matrix"); }

int nolsm_energy(nolsm_ctx* c, double* e_elec) try {
    if (!c || !e_elec) return NOLSM_EINVAL;
    if (!c->have_result || c->last_count_only) return fail(c, NOLSM_ESTATE, "no density matrix has been computed");
    cudaSetDevice(c->dev);
    if (int r = wait_result(c)) return r;
    const int64_t n = c->last_a1 - c->last_a0;
    std::vector<double> e(n);
    CU_TRY(c, cudaMemcpy(e.data(), c->d_e_atom + c->last_a0, 8 * n, cudaMemcpyDeviceToHost));
    double sum = 0;
    for (int64_t i = 0; i < n; ++i) sum += e[i];
    *e_elec = sum;
    int bits = 0;
    if (int r = engine_status_bits(c, &bits)) return r;
    if (bits & NOLSM_MAT_NOTSPD) return fail(c, NOLSM_ENOTSPD, "an S_sub inverse iteration failed (see nolsm_get_atom_stats)");
    if (bits & NOLSM_MAT_NOCONV) return fail(c, NOLSM_ENOCONV, "a sign iteration hit max_sign_iters (see nolsm_get_atom_stats)");
    return NOLSM_OK;
} catch (...) { return on_exception(c, "nolsm_energy"); }

int nolsm_electron_count(nolsm_ctx* c, double* n_elec, double* q_atom_out) try {
    if (!c || !n_elec) return NOLSM_EINVAL;
    if (!c->have_result || c->last_count_only) return fail(c, NOLSM_ESTATE, "no density matrix has been computed");
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
} catch (...) { return on_exception(c, "nolsm_electron_count"); }

int nolsm_electron_counts(nolsm_ctx* c, const double* mu, int n_mu, double* n_elec_out, double* e_out, void* cuda_stream) try {
    if (!c || !mu || !n_elec_out) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "nolsm_assemble has not been called");
    if (n_mu < 1 || n_mu > NOLSM_MAX_MU) return fail(c, NOLSM_EINVAL, "n_mu must be 1..8");
    if (!c->persist) return fail(c, NOLSM_ESTATE, "nolsm_electron_counts needs the persistent engine");
    if (int r = run(c, mu, n_mu, true, 0, c->n_atoms, nullptr, NOLSM_DTYPE_F64, cuda_stream)) return r;
    if (int r = wait_result(c)) return r;
    double acc[2 * NOLSM_MAX_MU];
    CU_TRY(c, cudaMemcpy(acc, c->d_mu_acc, sizeof(acc), cudaMemcpyDeviceToHost));
    for (int j = 0; j < n_mu; ++j) {
        n_elec_out[j] = acc[j];
        if (e_out) e_out[j] = acc[NOLSM_MAX_MU + j];
    }
    int bits = 0;
    if (int r = engine_status_bits(c, &bits)) return r;
    if (bits & NOLSM_MAT_NOTSPD) return fail(c, NOLSM_ENOTSPD, "an S_sub inverse iteration failed (see nolsm_get_atom_stats)");
    if (bits & NOLSM_MAT_NOCONV) return fail(c, NOLSM_ENOCONV, "a sign iteration hit max_sign_iters (see nolsm_get_atom_stats)");
    return NOLSM_OK;
} catch (...) { return on_exception(c, "nolsm_electron_counts"); }

int nolsm_find_mu(nolsm_ctx* c, double n_target, double mu_lo, double mu_hi, double tol_n, double tol_mu, int max_evals,
                  void* D_vals, int d_dtype, void* cuda_stream, double* mu_out, double* n_out, int* evals_out) try {
    if (!c || !D_vals || !mu_out) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "nolsm_assemble has not been called");
    if (!(mu_lo < mu_hi) || !(tol_n >= 0) || !(tol_mu >= 0)) return fail(c, NOLSM_EINVAL, "need mu_lo < mu_hi and tolerances >= 0");
    if (max_evals <= 0) max_evals = 40;
    // N(mu) = Tr(D(mu) S) never decreases with mu (it counts the generalised eigenvalues of every submatrix below mu,
    // weighted by their share in the atom's columns). Persistent engine: every pass over the atoms evaluates K trial mu
    // on the resident S_sub^-1 and A0 = S_sub^-1 H_sub (nolsm_electron_counts: only the sign chain and the traces repeat
    // per trial, PAPER.md:L149 / L155), so the bracket shrinks by K + 1 per pass; the last pass is one
    // nolsm_density_matrix call at the mu reported, which writes D_vals. Round engine: plain bisection.
    int evals = 0, rc_soft = NOLSM_OK;
    auto soften = [&](int r) { if (r == NOLSM_ENOCONV) { rc_soft = r; return (int)NOLSM_OK; } return r; };
    auto count_full = [&](double mu, double* n) -> int {
        int r = nolsm_density_matrix(c, mu, D_vals, d_dtype, cuda_stream);
        if (r) return r;
        ++evals;
        double e;
        if ((r = soften(nolsm_energy(c, &e)))) return r;       // flagged matrices are still written (nolsm.h)
        return nolsm_electron_count(c, n, nullptr);
    };
    const int K = c->persist ? std::max(1, std::min(c->opt.mu_trials > 0 ? c->opt.mu_trials : 1, NOLSM_MAX_MU)) : 1;
    double mu = mu_hi, n_mu = 0;
    int r;
    if (c->persist) {
        double ends[2] = {mu_lo, mu_hi}, ne[2];
        if ((r = soften(nolsm_electron_counts(c, ends, 2, ne, nullptr, cuda_stream)))) return r;
        evals += 2;
        n_mu = ne[1];
        if (ne[0] - tol_n > n_target || ne[1] + tol_n < n_target) {
            if (n_out) *n_out = ne[1];
            if (evals_out) *evals_out = evals;
            *mu_out = mu_hi;
            return fail(c, NOLSM_EINVAL, "nolsm_find_mu: the electron count is not bracketed by [mu_lo, mu_hi]");
        }
        bool hit = false;
        if (std::fabs(ne[0] - n_target) <= tol_n) { mu = mu_lo; n_mu = ne[0]; hit = true; }
        else if (std::fabs(ne[1] - n_target) <= tol_n) { mu = mu_hi; n_mu = ne[1]; hit = true; }
        while (!hit && evals < max_evals && (mu_hi - mu_lo) > tol_mu) {
            const int k = std::min(K, max_evals - evals);
            double tr[NOLSM_MAX_MU], nt[NOLSM_MAX_MU];
            for (int j = 0; j < k; ++j) tr[j] = mu_lo + (mu_hi - mu_lo) * (double)(j + 1) / (double)(k + 1);
            if ((r = soften(nolsm_electron_counts(c, tr, k, nt, nullptr, cuda_stream)))) return r;
            evals += k;
            // new bracket: the neighbouring trials around the target
            double lo = mu_lo, hi = mu_hi;
            for (int j = 0; j < k; ++j) {
                if (std::fabs(nt[j] - n_target) <= tol_n) { mu = tr[j]; n_mu = nt[j]; hit = true; break; }
                if (nt[j] < n_target) lo = tr[j]; else { hi = tr[j]; break; }
            }
            if (hit) break;
            mu_lo = lo; mu_hi = hi;
            mu = 0.5 * (mu_lo + mu_hi);
        }
        if (!hit) mu = 0.5 * (mu_lo + mu_hi);
        if ((r = count_full(mu, &n_mu))) return r;               // writes D(mu)
    } else {
        double n_lo, n_hi;
        if ((r = count_full(mu_lo, &n_lo))) return r;
        if ((r = count_full(mu_hi, &n_hi))) return r;
        mu = mu_hi; n_mu = n_hi;
        if (n_lo - tol_n > n_target || n_hi + tol_n < n_target) {
            if (n_out) *n_out = n_hi;
            if (evals_out) *evals_out = evals;
            *mu_out = mu_hi;
            return fail(c, NOLSM_EINVAL, "nolsm_find_mu: the electron count is not bracketed by [mu_lo, mu_hi]");
        }
        while (evals < max_evals && std::fabs(n_mu - n_target) > tol_n && (mu_hi - mu_lo) > tol_mu) {
            mu = 0.5 * (mu_lo + mu_hi);
            if ((r = count_full(mu, &n_mu))) return r;
            if (n_mu < n_target) mu_lo = mu; else mu_hi = mu;
        }
    }
    *mu_out = mu;
    if (n_out) *n_out = n_mu;
    if (evals_out) *evals_out = evals;
    if (rc_soft) return fail(c, rc_soft, "a sign iteration hit max_sign_iters during the mu search (see nolsm_get_atom_stats)");
    return NOLSM_OK;
} catch (...) { return on_exception(c, "nolsm_find_mu"); }

int nolsm_get_index_set(nolsm_ctx* c, int64_t atom, int32_t* atoms_out, int32_t* n_inout, int32_t* dim_out) try {
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
} catch (...) { return on_exception(c, "nolsm_get_index_set"); }

int nolsm_get_group(nolsm_ctx* c, int64_t atom, int32_t* members_out, int32_t* n_members_inout, int32_t* set_out,
                    int32_t* n_set_inout, int32_t* dim_out) try {
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
} catch (...) { return on_exception(c, "nolsm_get_group"); }

int nolsm_gather_submatrix(nolsm_ctx* c, int64_t atom, int which, int out_fp16, void* out_host) try {
    if (!c || !out_host || (which != 0 && which != 1)) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    if (atom < 0 || atom >= c->n_atoms) return fail(c, NOLSM_EINVAL, "atom out of range");
    cudaSetDevice(c->dev);
    if (c->have_result) { if (int r = wait_result(c)) return r; }
    // with combine the dense submatrix an atom is evaluated on is its group's (tight, dimension of nolsm_get_group)
    if (c->combined) return engine_gather(c, c->unit_of[atom], true, which, out_fp16, out_host);
    return engine_gather(c, atom, false, which, out_fp16, out_host);
} catch (...) { return on_exception(c, "nolsm_gather_submatrix"); }

// The gather without device allocations (static scratch array in engine.cu). It does not wait for the last
// density_matrix call: it reads only the pattern and the H0 / S values and writes only the scratch array and `out`.
int nolsm_gather_submatrix_noalloc(nolsm_ctx* c, int64_t atom, int which, void* out, void* cuda_stream) try {
    if (!c || !out || (which != 0 && which != 1)) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    if (atom < 0 || atom >= c->n_atoms) return fail(c, NOLSM_EINVAL, "atom out of range");
    cudaSetDevice(c->dev);
    return engine_gather_noalloc(c, c->combined ? c->unit_of[atom] : atom, which, out, (cudaStream_t)cuda_stream);
} catch (...) { return on_exception(c, "nolsm_gather_submatrix_noalloc"); }

int nolsm_get_atom_stats(nolsm_ctx* c, int64_t a0, int64_t count, int32_t* dims, int32_t* inv_iters, int32_t* sign_iters,
                         int32_t* status, int32_t* gemms, float* residual, double* e_atom) try {
    if (!c) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    if (a0 < 0 || count < 0 || a0 + count > c->n_atoms) return fail(c, NOLSM_EINVAL, "range");
    cudaSetDevice(c->dev);
    if (c->have_result) { if (int r = wait_result(c)) return r; }
    return engine_atom_stats(c, a0, count, dims, inv_iters, sign_iters, status, gemms, residual, e_atom);
} catch (...) { return on_exception(c, "nolsm_get_atom_stats"); }

int nolsm_get_stats(nolsm_ctx* c, nolsm_stats* out) try {
    if (!c || !out) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    memset(out, 0, sizeof(*out));
    out->n_atoms = c->n_atoms;
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
        cudaSetDevice(c->dev);
        if (int r = wait_result(c)) return r;
        return engine_stats(c, out);
    }
    return NOLSM_OK;
} catch (...) { return on_exception(c, "nolsm_get_stats"); }

int nolsm_get_profile(nolsm_ctx* c, double* out, int n) try {
    if (!c || !out || n < NOLSM_PROFILE_LEN) return NOLSM_EINVAL;
    if (!c->have_result) return fail(c, NOLSM_ESTATE, "no density matrix has been computed");
    cudaSetDevice(c->dev);
    if (int r = wait_result(c)) return r;
    return engine_profile(c, out);
} catch (...) { return on_exception(c, "nolsm_get_profile"); }

int nolsm_get_engine_counters(nolsm_ctx* c, double* out, int n) try {
    if (!c || !out || n < NOLSM_COUNTERS_LEN) return NOLSM_EINVAL;
    if (!c->have_result) return fail(c, NOLSM_ESTATE, "no density matrix has been computed");
    cudaSetDevice(c->dev);
    if (int r = wait_result(c)) return r;
    return engine_counters(c, out);
} catch (...) { return on_exception(c, "nolsm_get_engine_counters"); }

int nolsm_side_task_bandwidth(nolsm_ctx* c, int which, int reps, double* ms_out, double* bytes_out) try {
    if (!c || !ms_out || !bytes_out || (which != 0 && which != 1) || reps < 1) return NOLSM_EINVAL;
    if (!c->assembled) return fail(c, NOLSM_ESTATE, "not assembled");
    cudaSetDevice(c->dev);
    if (c->have_result) { if (int r = wait_result(c)) return r; }
    return engine_side_bandwidth(c, which, reps, ms_out, bytes_out);
} catch (...) { return on_exception(c, "nolsm_side_task_bandwidth"); }

}  // extern "C"
