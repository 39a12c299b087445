// Host-side setup: cell grid / octree and the task list.
// Plain C++ (no device code); written independently of the oracle's builders and cross-checked against them
// in tests/test_host_side.py.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "internal.h"

using namespace sph;

namespace {

struct Node { uint64_t lo, hi; double o[3]; double w; uint32_t depth; };

inline int octant_of(const double* x, const double* o, double w) {
    const double half = 0.5 * w;
    return (x[0] >= o[0] + half ? 4 : 0) | (x[1] >= o[1] + half ? 2 : 0) | (x[2] >= o[2] + half ? 1 : 0);
}

// smallest periodic gap between the intervals [a, a+wa] and [b, b+wb]; shift = image offset applied to b
inline double gap_1d(double a, double wa, double b, double wb, double box, double* shift, double* runner_up) {
    double g[3];
    for (int k = 0; k < 3; ++k) {
        const double s = (k - 1) * box;
        const double left = (b + s) - (a + wa), right = a - (b + s + wb);
        g[k] = std::max(0.0, std::max(left, right));
    }
    int best = 0;
    for (int k = 1; k < 3; ++k) if (g[k] < g[best]) best = k;
    double second = 1e300;
    for (int k = 0; k < 3; ++k) if (k != best) second = std::min(second, g[k]);
    *shift = (best - 1) * box;
    *runner_up = second;
    return g[best];
}

// Order inside a cell (reading C26): ascending Morton code of the position on a 32^3 sub-grid of the cell, ties in
// input order.  Spatially compact runs of particles are what lets the interaction loops drop whole chunks of a
// neighbouring cell before any distance test.  spread5: bits b of a 5-bit number go to bits 3b.
inline uint32_t spread5(uint32_t v) { return (v & 1u) | (v & 2u) << 2 | (v & 4u) << 4 | (v & 8u) << 6 | (v & 16u) << 8; }
inline uint32_t sub_cell_code(const double* x, const double* o, double w) {
    uint32_t q[3];
    for (int d = 0; d < 3; ++d) {
        const double f = std::floor((x[d] - o[d]) / w * 32.0);
        q[d] = f < 0.0 ? 0u : (f > 31.0 ? 31u : (uint32_t)f);
    }
    return spread5(q[0]) << 2 | spread5(q[1]) << 1 | spread5(q[2]);
}
// idx[lo, hi) -> Morton order inside the cell; scratch holds (code << 32 | position) so that one plain sort is stable
void order_inside_cell(const double* x3, uint64_t* idx, uint64_t lo, uint64_t hi, const double* o, double w, std::vector<uint64_t>& scratch,
                       std::vector<uint64_t>& tmp) {
    const uint64_t cnt = hi - lo;
    if (cnt < 2) return;
    scratch.resize(cnt);
    tmp.resize(cnt);
    for (uint64_t k = 0; k < cnt; ++k) scratch[k] = (uint64_t)sub_cell_code(x3 + 3 * idx[lo + k], o, w) << 32 | k;
    std::sort(scratch.begin(), scratch.end());
    for (uint64_t k = 0; k < cnt; ++k) tmp[k] = idx[lo + (scratch[k] & 0xFFFFFFFFull)];
    std::copy(tmp.begin(), tmp.end(), idx + lo);
}

}  // namespace

extern "C" {

int32_t sph_free(void* p) { std::free(p); return SPH_OK; }

int32_t sph_cells_build_grid(const double* x3, uint64_t n, uint32_t cpd, double box, uint64_t* perm_out, sph_cell* cells_out) {
    if (!x3 || !perm_out || !cells_out) return fail(SPH_ERR_INVALID_ARG, "NULL argument");
    if (cpd == 0 || cpd > 1024 || !(box > 0)) return fail(SPH_ERR_INVALID_ARG, "cells_per_dim %u, box %g", cpd, box);
    SPH_API_BEGIN
    const uint64_t nc = (uint64_t)cpd * cpd * cpd;
    std::vector<uint32_t> key(n);
    std::vector<uint64_t> head(nc + 1, 0);
    for (uint64_t p = 0; p < n; ++p) {
        uint32_t c = 0;
        for (int d = 0; d < 3; ++d) {
            const double xv = x3[3 * p + d];
            if (!(xv >= 0.0 && xv < box)) return fail(SPH_ERR_RANGE, "particle %llu: x[%d] = %.17g outside [0, %g)", (unsigned long long)p, d, xv, box);
            const uint32_t k = std::min<uint32_t>(cpd - 1, (uint32_t)std::floor(xv / box * cpd));
            c = c * cpd + k;
        }
        key[p] = c;
        ++head[c + 1];
    }
    for (uint64_t c = 0; c < nc; ++c) head[c + 1] += head[c];
    const double w = box / cpd;
    for (uint64_t c = 0; c < nc; ++c) {
        sph_cell& ce = cells_out[c];
        ce.first = head[c];
        ce.count = (uint32_t)(head[c + 1] - head[c]);
        ce.pad = 0;
        ce.width = w;
        ce.origin[0] = (double)(c / ((uint64_t)cpd * cpd)) * w;
        ce.origin[1] = (double)((c / cpd) % cpd) * w;
        ce.origin[2] = (double)(c % cpd) * w;
    }
    std::vector<uint64_t> cursor(head.begin(), head.end() - 1);
    for (uint64_t p = 0; p < n; ++p) perm_out[cursor[key[p]]++] = p;   // counting sort: stable
    std::vector<uint64_t> scratch, tmp;
    for (uint64_t c = 0; c < nc; ++c) order_inside_cell(x3, perm_out, head[c], head[c + 1], cells_out[c].origin, w, scratch, tmp);
    return SPH_OK;
    SPH_API_END
}

int32_t sph_cells_build_octree(const double* x3, const float* h, uint64_t n, uint32_t max_per_leaf, double box, uint64_t* perm_out,
                               sph_cell** cells_out, uint32_t* n_cells_out) {
    if (!x3 || !h || !perm_out || !cells_out || !n_cells_out) return fail(SPH_ERR_INVALID_ARG, "NULL argument");
    if (max_per_leaf == 0 || !(box > 0)) return fail(SPH_ERR_INVALID_ARG, "max_per_leaf %u, box %g", max_per_leaf, box);
    SPH_API_BEGIN
    for (uint64_t p = 0; p < n; ++p)
        for (int d = 0; d < 3; ++d)
            if (!(x3[3 * p + d] >= 0.0 && x3[3 * p + d] < box)) return fail(SPH_ERR_RANGE, "particle %llu outside the box", (unsigned long long)p);
    std::vector<uint64_t> idx(n), tmp(n);
    for (uint64_t p = 0; p < n; ++p) idx[p] = p;
    std::vector<sph_cell> leaves;
    std::vector<Node> stack;
    stack.push_back(Node{0, n, {0, 0, 0}, box, 0});
    while (!stack.empty()) {
        const Node nd = stack.back();
        stack.pop_back();
        const uint64_t cnt = nd.hi - nd.lo;
        if (cnt == 0) continue;
        bool split = cnt > max_per_leaf && nd.depth < 20;
        uint64_t occ[8] = {};
        if (split) {
            float hm[8] = {};
            for (uint64_t k = nd.lo; k < nd.hi; ++k) {
                const int o = octant_of(x3 + 3 * idx[k], nd.o, nd.w);
                ++occ[o];
                hm[o] = std::max(hm[o], h[idx[k]]);
            }
            for (int o = 0; o < 8; ++o)
                if (occ[o] && !(0.5 * nd.w >= 2.0 * (double)hm[o])) split = false;   // a child would be narrower than 2 hmax
        }
        if (!split) {
            sph_cell ce;
            ce.first = nd.lo; ce.count = (uint32_t)cnt; ce.pad = 0; ce.width = nd.w;
            ce.origin[0] = nd.o[0]; ce.origin[1] = nd.o[1]; ce.origin[2] = nd.o[2];
            leaves.push_back(ce);
            continue;
        }
        uint64_t begin[9];
        begin[0] = nd.lo;
        for (int o = 0; o < 8; ++o) begin[o + 1] = begin[o] + occ[o];
        uint64_t cur[8];
        for (int o = 0; o < 8; ++o) cur[o] = begin[o];
        for (uint64_t k = nd.lo; k < nd.hi; ++k) tmp[cur[octant_of(x3 + 3 * idx[k], nd.o, nd.w)]++] = idx[k];   // stable
        std::copy(tmp.begin() + nd.lo, tmp.begin() + nd.hi, idx.begin() + nd.lo);
        for (int o = 7; o >= 0; --o) {   // push in reverse so that octant 0 is processed first (depth-first order)
            Node ch{begin[o], begin[o + 1], {nd.o[0] + ((o >> 2) & 1) * 0.5 * nd.w, nd.o[1] + ((o >> 1) & 1) * 0.5 * nd.w,
                                            nd.o[2] + (o & 1) * 0.5 * nd.w}, 0.5 * nd.w, nd.depth + 1};
            stack.push_back(ch);
        }
    }
    std::vector<uint64_t> scratch;
    for (const sph_cell& ce : leaves) order_inside_cell(x3, idx.data(), ce.first, ce.first + ce.count, ce.origin, ce.width, scratch, tmp);
    std::copy(idx.begin(), idx.end(), perm_out);
    sph_cell* out = (sph_cell*)std::malloc(std::max<size_t>(1, leaves.size()) * sizeof(sph_cell));
    if (!out) return fail(SPH_ERR_ALLOC, "cells allocation failed");
    std::memcpy(out, leaves.data(), leaves.size() * sizeof(sph_cell));
    *cells_out = out;
    *n_cells_out = (uint32_t)leaves.size();
    return SPH_OK;
    SPH_API_END
}

int32_t sph_tasks_build(const sph_cell* cells, const float* hmax, uint32_t n_cells, double box, sph_task** tasks_out, uint64_t* n_self_out,
                        uint64_t* n_pair_out) {
    if (!cells || !hmax || !tasks_out || n_cells == 0) return fail(SPH_ERR_INVALID_ARG, "NULL argument or no cells");
    SPH_API_BEGIN
    double reach = 0;   // largest cut-off any pair can have
    for (uint32_t c = 0; c < n_cells; ++c) {
        reach = std::max(reach, 2.0 * (double)hmax[c]);
        // a cell must not see its own periodic image: the self task is not periodic
        if (cells[c].count && !(box - cells[c].width >= 2.0 * (double)hmax[c]))
            return fail(SPH_ERR_RANGE, "cell %u (width %g, 2 hmax %g) interacts with its own periodic image in a box of %g", c, cells[c].width,
                        2.0 * (double)hmax[c], box);
    }
    // bin the cells on a uniform grid; a cell is listed in every bin its box overlaps
    int nb = (int)std::min(64.0, std::max(1.0, std::floor(box / std::max(reach, 1e-9))));
    nb = std::min(nb, std::max(1, (int)std::cbrt((double)n_cells)));
    const double bw = box / nb;
    auto bin_range = [&](double lo, double hi, int* b0, int* b1) {   // inclusive, may run outside [0, nb): wrap on use
        *b0 = (int)std::floor(lo / bw);
        *b1 = (int)std::floor(hi / bw);
        if (*b1 - *b0 >= nb) { *b0 = 0; *b1 = nb - 1; }
    };
    std::vector<std::vector<uint32_t>> bins((size_t)nb * nb * nb);
    for (uint32_t c = 0; c < n_cells; ++c) {
        int r0[3], r1[3];
        for (int d = 0; d < 3; ++d) bin_range(cells[c].origin[d], cells[c].origin[d] + cells[c].width * (1 - 1e-12), &r0[d], &r1[d]);
        for (int a = r0[0]; a <= r1[0]; ++a) for (int b = r0[1]; b <= r1[1]; ++b) for (int e = r0[2]; e <= r1[2]; ++e)
            bins[((size_t)((a % nb + nb) % nb) * nb + ((b % nb + nb) % nb)) * nb + ((e % nb + nb) % nb)].push_back(c);
    }
    std::vector<sph_task> tasks;
    tasks.reserve((size_t)n_cells * 14);
    for (uint32_t c = 0; c < n_cells; ++c) {
        sph_task t;
        t.ci = (int32_t)c; t.cj = -1;
        for (int d = 0; d < 3; ++d) t.frame_i[d] = t.frame_j[d] = cells[c].origin[d];
        tasks.push_back(t);
    }
    std::vector<uint32_t> stamp(n_cells, UINT32_MAX), cand;
    for (uint32_t a = 0; a < n_cells; ++a) {
        cand.clear();
        int r0[3], r1[3];
        for (int d = 0; d < 3; ++d) bin_range(cells[a].origin[d] - reach, cells[a].origin[d] + cells[a].width + reach, &r0[d], &r1[d]);
        for (int i = r0[0]; i <= r1[0]; ++i) for (int j = r0[1]; j <= r1[1]; ++j) for (int k = r0[2]; k <= r1[2]; ++k) {
            const auto& lst = bins[((size_t)((i % nb + nb) % nb) * nb + ((j % nb + nb) % nb)) * nb + ((k % nb + nb) % nb)];
            for (uint32_t b : lst)
                if (b > a && stamp[b] != a) { stamp[b] = a; cand.push_back(b); }
        }
        std::sort(cand.begin(), cand.end());
        for (uint32_t b : cand) {
            const double cut = std::max(2.0 * (double)hmax[a], 2.0 * (double)hmax[b]);
            double g2 = 0, shift[3];
            bool second_image_in_reach = false;
            for (int d = 0; d < 3; ++d) {
                double ru;
                const double g = gap_1d(cells[a].origin[d], cells[a].width, cells[b].origin[d], cells[b].width, box, &shift[d], &ru);
                g2 += g * g;
                second_image_in_reach |= ru < cut;
            }
            if (!(std::sqrt(g2) < cut)) continue;
            if (second_image_in_reach)
                return fail(SPH_ERR_RANGE, "cells %u and %u interact through two periodic images (box too small for the cut-off)", a, b);
            sph_task t;
            t.ci = (int32_t)a; t.cj = (int32_t)b;
            for (int d = 0; d < 3; ++d) { t.frame_i[d] = cells[a].origin[d]; t.frame_j[d] = cells[a].origin[d] - shift[d]; }
            tasks.push_back(t);
        }
    }
    sph_task* out = (sph_task*)std::malloc(tasks.size() * sizeof(sph_task));
    if (!out) return fail(SPH_ERR_ALLOC, "task allocation failed");
    std::memcpy(out, tasks.data(), tasks.size() * sizeof(sph_task));
    *tasks_out = out;
    if (n_self_out) *n_self_out = n_cells;
    if (n_pair_out) *n_pair_out = tasks.size() - n_cells;
    return SPH_OK;
    SPH_API_END
}

}  // extern "C"
