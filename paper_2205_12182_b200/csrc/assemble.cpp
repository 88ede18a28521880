// nolsm_assemble (a0): validation of the block-CSR pattern, index sets N(i), dimensions, the optional
// max-abs filter (C-1), the units of the submatrix combination (grouping.cpp) and the uploads of the index
// data. Host integer logic; the workspace plan and everything that touches kernels is engine.cu (engine_plan).
#include <atomic>

#include "ctx.h"

using namespace nolsm_host;

extern "C" {

int nolsm_assemble(nolsm_ctx* c, int64_t n_atoms, const int32_t* atom_nb, const int64_t* row_ptr,
                   const int32_t* col_idx, const void* H0_vals, const void* S_vals, int val_dtype, void* cuda_stream) try {
    if (!c) return NOLSM_EINVAL;
    if (n_atoms <= 0 || !atom_nb || !row_ptr || !col_idx || !H0_vals || !S_vals)
        return fail(c, NOLSM_EINVAL, "null pointer or n_atoms <= 0");
    if (val_dtype != NOLSM_DTYPE_F64 && val_dtype != NOLSM_DTYPE_F32) return fail(c, NOLSM_EINVAL, "bad val_dtype");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaSetDevice(c->dev);
    auto t_prev = std::chrono::steady_clock::now();
    auto lap = [&](const char* what) {
        if (!verbose(1)) return;
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
        if ((r = engine_block_keep(c, d_keep, s))) return r;
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
    build_units(c, c->combined ? c->opt.combine : 0, std::min(c->opt.combine_max_dim, 4096), c->opt.combine_max_members,
                c->opt.combine_max_candidates);
    lap("units (grouping)");
    int max_n = 0, min_n = 1 << 30, max_nset = 0, max_nbi = 0;
    for (int64_t i = 0; i < n_atoms; ++i) max_nbi = std::max(max_nbi, c->atom_nb[i]);
    for (int64_t u = 0; u < c->n_units; ++u) {
        max_n = std::max(max_n, c->udim[u]);
        min_n = std::min(min_n, c->udim[u]);
        max_nset = std::max<int>(max_nset, (int)(c->uset_ptr[u + 1] - c->uset_ptr[u]));
    }
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
    if ((r = engine_plan(c, s))) return r;
    CU_TRY(c, cudaStreamSynchronize(s));
    lap("workspace, maps, engine");
    c->assembled = true;
    return NOLSM_OK;
} catch (...) { return on_exception(c, "nolsm_assemble"); }

}  // extern "C"
