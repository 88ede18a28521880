// Submatrix combination (Eq. 9 / Eq. 10; C-19): which atoms share one dense submatrix.
// Host integer arithmetic only: the grouping is reproducible bit for bit by any restatement of DESIGN.md C-19.
#include "ctx.h"

namespace nolsm_host {

// Predicted cost of evaluating the matrix function on a submatrix of dimension n.
//   mode 1 (Eq. 9):  n^3, the FLOP of a dense multiplication.
//   mode 2 (Eq. 10): the predicted runtime n^3 / r(n), r(n) = the measured multiplication rate of the GPU
//     "measured for different matrix sizes n and interpolated" (L89): the table set with nolsm_set_perf_table (integers:
//     dimensions and GFLOP/s), linear interpolation between neighbouring entries, constant outside the table. In
//     integers: r = (r_k (n_{k+1} - n) + r_{k+1} (n - n_k)) / (n_{k+1} - n_k), cost = 10^6 n^3 / r (floor divisions of
//     non-negative numbers). Without a table: the tile-step count of the engine, ceil(n16/256)^2 ceil(n16/64) (the time
//     of a multiplication in 256 x 256 x 64 tile steps), a model that the CPU tests compare with the
//     measured table.
int64_t perf_rate(const std::vector<int64_t>& tn, const std::vector<int64_t>& tr, int64_t n) {
    const size_t m = tn.size();
    if (n <= tn[0]) return tr[0];
    if (n >= tn[m - 1]) return tr[m - 1];
    size_t k = (size_t)(std::upper_bound(tn.begin(), tn.end(), n) - tn.begin()) - 1;      // tn[k] <= n < tn[k + 1]
    return (tr[k] * (tn[k + 1] - n) + tr[k + 1] * (n - tn[k])) / (tn[k + 1] - tn[k]);
}

int64_t combine_cost(const nolsm_ctx* c, int64_t n, int mode) {
    if (mode == 1) return n * n * n;
    if (!c->pn_n.empty()) return (int64_t)1000000 * n * n * n / perf_rate(c->pn_n, c->pn_rate, n);
    const int64_t n16 = (n + 15) / 16 * 16, t = (n16 + 255) / 256;
    return t * t * ((n16 + 63) / 64);
}

// Builds the units of the context from the per-atom index sets: greedy groups (mode 1 / 2) or one atom per unit (mode 0).
void build_units(nolsm_ctx* c, int mode, int max_dim, int max_members, int max_cand) {
    const int64_t n_at = c->n_atoms;
    const int32_t* nb = c->atom_nb.data();
    c->unit_ptr.assign(1, 0); c->unit_mem.clear(); c->uset_ptr.assign(1, 0); c->uset_atom.clear(); c->uset_off.clear(); c->udim.clear();
    c->unit_of.assign(n_at, -1); c->upos.assign(n_at, 0);
    auto t_prev = std::chrono::steady_clock::now();
    auto lap = [&](const char* what) {
        if (!verbose(2)) return;
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
                if (combine_cost(c, n_u, mode) < combine_cost(c, n_g, mode) + combine_cost(c, c->dim[j], mode)) {
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

}  // namespace nolsm_host
