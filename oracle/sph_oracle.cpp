// ORACLE -- test infrastructure, NOT the product.
//
// A plain, slow, obviously-correct CPU restatement of the data-parallel hot path
// of arxiv/paper_2606_23891 ("Memory Layouts for GPU-Data Transfer Buffering in
// SPH"): cells -> tasks -> pack -> density loop -> unpack -> ghost -> pack ->
// force loop -> unpack.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference leg may build, load or call this file.  It
// shares no code, header, table or helper with the CUDA path
// (paper_2606_23891_b200/csrc); the record and struct layouts are restated here.
//
// What fixes each step (PAPER.md = /root/reference/PAPER.md; "reading Cn" =
// DESIGN.md section "Readings of the paper"):
//   particle record ........ PAPER.md:47-58 Table 1 + BASELINE.json:configs[0]   (C16)
//   cells .................. PAPER.md:66   (particles sorted by cell; inside a cell by the Morton code of
//                            their position, reading C26)
//   tasks / bundles ........ PAPER.md:70, 76
//   pack ................... PAPER.md:78, 102 ("only the required quantities are buffered",
//                            "coordinates shifted to facilitate periodic boundary conditions") (C6, C7)
//   density / force loops .. PAPER.md:39-41; the paper prints no formula and cites Price 2012:
//                            cubic spline, support 2h, grad-h terms, Monaghan viscosity (C1, C2, C9-C13)
//   unpack ................. PAPER.md:82 ("performs all required reductions")  (C8)
//   ghost .................. PAPER.md:62 (linear update kernels)               (C12)
//   gradient loop, Balsara . PAPER.md:41, Table 1 columns p-g / u-g / p-f (47-58)  (C34; next-scope row f2)
//
// Arithmetic: record values are f32 (Table 1); the loops promote them to f64,
// accumulate in f64 and round once to f32.  pack does one f64 subtraction and
// one round-to-nearest conversion per coordinate.  unpack adds in f32, in
// ascending task order, side i before side j.  Compile with -ffp-contract=off.
//
// Parity pins: tests/test_oracle_pins.py (every function below is pinned, the test-support functions orc_compare_blocks and
// orc_flag_cutoff_pairs and the floor of balsara() included since round 3; none
// is "parity unpinned" except v_sig exactly at the cut-off, reading C31).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

const double kPi = 3.14159265358979323846264338327950288;

// ---- the canonical particle (C16): natural C alignment gives the offsets below ----
struct Part {
    double x[3];
    float v[3];
    float a[3];
    float mass, h, u, du_dt;
    float rho, rho_dh, wcount, wcount_dh;
    float div_v;
    float rot_v[3];
    float P, cs, v_sig;
    float pad0;
    int64_t id;
    int8_t time_bin;
    int8_t pad1[7];
};
static_assert(sizeof(Part) == 128, "canonical particle is 128 bytes");
static_assert(offsetof(Part, v) == 24 && offsetof(Part, a) == 36 && offsetof(Part, mass) == 48 &&
              offsetof(Part, rho) == 64 && offsetof(Part, div_v) == 80 && offsetof(Part, rot_v) == 84 &&
              offsetof(Part, P) == 96 && offsetof(Part, v_sig) == 104 && offsetof(Part, id) == 112 &&
              offsetof(Part, time_bin) == 120, "offsets of reading C16");

struct Cell {            // cell c owns particles [first, first+count)
    uint64_t first;
    uint32_t count;
    uint32_t pad;
    double origin[3];
    double width;
};
static_assert(sizeof(Cell) == 48, "");

struct Task {            // one loop step on one cell (cj = -1) or one cell pair
    int32_t ci, cj;
    double frame_i[3];   // side-i coordinates are packed relative to this point
    double frame_j[3];   // side-j ditto; includes the periodic image shift
};
static_assert(sizeof(Task) == 56, "");

enum Field { X, V, A, MASS, H, U, DU_DT, RHO, RHO_DH, WCOUNT, WCOUNT_DH, DIV_V, ROT_V, PRES, CS, V_SIG, ID, TIME_BIN, NFIELDS };
const uint32_t FLAG_X_REL_F32 = 1u;
enum Mode { MODE_REDUCE = 0, MODE_ASSIGN = 1 };

int g_threads = 1;

// One entry of an attribute set: components [comp0, comp0+ncomp) of a field.
struct Attr { int32_t field, comp0, ncomp; };

// bytes one component of `field` occupies in a record
int comp_bytes(int field, uint32_t flags) {
    if (field == X) return (flags & FLAG_X_REL_F32) ? 4 : 8;
    if (field == ID) return 8;
    return 4;   // f32 members; time_bin: 4 bytes, value in byte 0, bytes 1-3 zero
}
int field_ncomp(int field) { return (field == X || field == V || field == A || field == ROT_V) ? 3 : 1; }

float* f32_member(Part& p, int field) {
    switch (field) {
        case V: return p.v;            case A: return p.a;            case MASS: return &p.mass;
        case H: return &p.h;           case U: return &p.u;           case DU_DT: return &p.du_dt;
        case RHO: return &p.rho;       case RHO_DH: return &p.rho_dh; case WCOUNT: return &p.wcount;
        case WCOUNT_DH: return &p.wcount_dh; case DIV_V: return &p.div_v; case ROT_V: return p.rot_v;
        case PRES: return &p.P;        case CS: return &p.cs;         case V_SIG: return &p.v_sig;
        default: return nullptr;
    }
}

int record_bytes(const Attr* attrs, int n_attr, uint32_t flags) {
    int b = 0;
    for (int k = 0; k < n_attr; ++k) b += attrs[k].ncomp * comp_bytes(attrs[k].field, flags);
    return b;
}

bool attrs_valid(const Attr* attrs, int n_attr) {
    bool seen[NFIELDS][3] = {};
    for (int k = 0; k < n_attr; ++k) {
        const Attr& a = attrs[k];
        if (a.field < 0 || a.field >= NFIELDS || a.comp0 < 0 || a.ncomp < 1 || a.comp0 + a.ncomp > field_ncomp(a.field)) return false;
        for (int c = a.comp0; c < a.comp0 + a.ncomp; ++c) {
            if (seen[a.field][c]) return false;
            seen[a.field][c] = true;
        }
    }
    return true;
}

uint64_t round_up(uint64_t v, uint64_t m) { return (v + m - 1) / m * m; }

// Buffer layout (C7): for each task in order: side-i block, then side-j block (pair only);
// a block is `count` records in store order and starts at the next multiple of 128 bytes.
// off[2*t], off[2*t+1] = byte offsets of the two blocks (off[2t+1] = UINT64_MAX for self tasks).
uint64_t block_offsets(const Cell* cells, const Task* tasks, int64_t n_tasks, int rec_bytes, uint64_t* off) {
    uint64_t run = 0;
    for (int64_t t = 0; t < n_tasks; ++t) {
        off[2 * t] = run;
        run = round_up(run + (uint64_t)cells[tasks[t].ci].count * rec_bytes, 128);
        if (tasks[t].cj >= 0) {
            off[2 * t + 1] = run;
            run = round_up(run + (uint64_t)cells[tasks[t].cj].count * rec_bytes, 128);
        } else {
            off[2 * t + 1] = UINT64_MAX;
        }
    }
    return run;
}

// ---- the kernel function (C2): Monaghan M4 cubic spline, support 2h, sigma = 1/pi ----
double w_of_q(double q) {
    if (q < 1.0) return 1.0 - 1.5 * q * q + 0.75 * q * q * q;
    if (q < 2.0) { double t = 2.0 - q; return 0.25 * t * t * t; }
    return 0.0;
}
double dw_of_q(double q) {
    if (q < 1.0) return -3.0 * q + 2.25 * q * q;
    if (q < 2.0) { double t = 2.0 - q; return -0.75 * t * t; }
    return 0.0;
}
double W(double r, double h) { return w_of_q(r / h) / (kPi * h * h * h); }
double dW_dh(double r, double h) { double q = r / h; return -(3.0 * w_of_q(q) + q * dw_of_q(q)) / (kPi * h * h * h * h); }
double dW_dr(double r, double h) { return dw_of_q(r / h) / (kPi * h * h * h * h); }

// ---- density partial sums of one target against one source block (reading step 6) ----
// records: DENSITY_IN = [xr0 xr1 xr2 h mass] f32
void density_block(const float* tgt, uint32_t n_t, const float* src, uint32_t n_s, float* out) {
    for (uint32_t i = 0; i < n_t; ++i) {
        const float* ri = tgt + 5 * i;
        const double hi = ri[3];
        double rho = 0, rho_dh = 0, wc = 0, wc_dh = 0;
        for (uint32_t j = 0; j < n_s; ++j) {          // self tasks: src == tgt, j == i included (C9)
            const float* rj = src + 5 * j;
            const double dx = (double)ri[0] - (double)rj[0], dy = (double)ri[1] - (double)rj[1], dz = (double)ri[2] - (double)rj[2];
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (r2 < 4.0 * hi * hi) {                  // strict < (C10)
                const double r = std::sqrt(r2), mj = rj[4];
                const double wv = W(r, hi), dv = dW_dh(r, hi);
                rho += mj * wv; rho_dh += mj * dv; wc += wv; wc_dh += dv;
            }
        }
        float* o = out + 4 * i;                       // DENSITY_OUT = [rho rho_dh wcount wcount_dh]
        o[0] = (float)rho; o[1] = (float)rho_dh; o[2] = (float)wc; o[3] = (float)wc_dh;
    }
}

// ---- force partial sums (reading step 9) ----
// records: FORCE_IN = [xr0 xr1 xr2 h mass rho rho_dh v0 v1 v2 u P cs] f32
void force_block(const float* tgt, uint32_t n_t, const float* src, uint32_t n_s, bool self, float* out,
                 double alpha, double beta) {
    for (uint32_t i = 0; i < n_t; ++i) {
        const float* ri = tgt + 13 * i;
        const double hi = ri[3], rhoi = ri[5], rho_dhi = ri[6], Pi = ri[11], ci = ri[12];
        const double omega_i = 1.0 + hi * rho_dhi / (3.0 * rhoi);
        const double Ai = Pi / (omega_i * rhoi * rhoi);
        double ax = 0, ay = 0, az = 0, dudt = 0, vsig = 0;
        for (uint32_t j = 0; j < n_s; ++j) {
            if (self && j == i) continue;
            const float* rj = src + 13 * j;
            const double hj = rj[3], mj = rj[4], rhoj = rj[5], rho_dhj = rj[6], Pj = rj[11], cj = rj[12];
            const double dx = (double)ri[0] - (double)rj[0], dy = (double)ri[1] - (double)rj[1], dz = (double)ri[2] - (double)rj[2];
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double hcut = std::max(2.0 * hi, 2.0 * hj);
            if (r2 > 0.0 && r2 < hcut * hcut) {        // coincident particles are skipped (C28)
                const double r = std::sqrt(r2);
                const double ex = dx / r, ey = dy / r, ez = dz / r;
                const double omega_j = 1.0 + hj * rho_dhj / (3.0 * rhoj);
                const double Aj = Pj / (omega_j * rhoj * rhoj);
                const double Gi = dW_dr(r, hi), Gj = dW_dr(r, hj), Gbar = 0.5 * (Gi + Gj);
                const double vr = ((double)ri[7] - (double)rj[7]) * ex + ((double)ri[8] - (double)rj[8]) * ey + ((double)ri[9] - (double)rj[9]) * ez;
                const double mu = std::min(0.0, vr);
                const double vs = ci + cj - beta * mu;
                const double Pi_visc = -0.5 * alpha * vs * mu / (0.5 * (rhoi + rhoj));
                const double fr = -mj * (Ai * Gi + Aj * Gj + Pi_visc * Gbar);
                ax += fr * ex; ay += fr * ey; az += fr * ez;
                dudt += mj * (Ai * Gi + 0.5 * Pi_visc * Gbar) * vr;
                vsig = std::max(vsig, vs);
            }
        }
        float* o = out + 5 * i;                       // FORCE_OUT = [a0 a1 a2 du_dt v_sig]
        o[0] = (float)ax; o[1] = (float)ay; o[2] = (float)az; o[3] = (float)dudt; o[4] = (float)vsig;
    }
}

// ---- gradient partial sums ("a third gradient loop between the density and the force loops"; reading C34) ----
// records: GRADIENT_IN = [xr0 xr1 xr2 v0 v1 v2 mass h u rho] f32 (Table 1, column p-g: x, v, mass, h, u, rho; u is packed as
// the table says, its consumer -- Sphenix' diffusion term -- is not part of this reading).
// For instance i over j != i with 0 < r < 2 h_i:  g = (m_j / rho_j) dW/dr(r, h_i),  e = (x_i - x_j) / r,  dv = v_j - v_i
//   div_v += g (dv . e)        rot_v += g (e x dv)
// GRADIENT_OUT = [div_v rot_v0 rot_v1 rot_v2].
void gradient_block(const float* tgt, uint32_t n_t, const float* src, uint32_t n_s, bool self, float* out) {
    for (uint32_t i = 0; i < n_t; ++i) {
        const float* ri = tgt + 10 * i;
        const double hi = ri[7];
        double div = 0, rx = 0, ry = 0, rz = 0;
        for (uint32_t j = 0; j < n_s; ++j) {
            if (self && j == i) continue;
            const float* rj = src + 10 * j;
            const double dx = (double)ri[0] - (double)rj[0], dy = (double)ri[1] - (double)rj[1], dz = (double)ri[2] - (double)rj[2];
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (r2 > 0.0 && r2 < 4.0 * hi * hi) {
                const double r = std::sqrt(r2);
                const double ex = dx / r, ey = dy / r, ez = dz / r;
                const double g = (double)rj[6] / (double)rj[9] * dW_dr(r, hi);
                const double dvx = (double)rj[3] - (double)ri[3], dvy = (double)rj[4] - (double)ri[4], dvz = (double)rj[5] - (double)ri[5];
                div += g * (dvx * ex + dvy * ey + dvz * ez);
                rx += g * (ey * dvz - ez * dvy); ry += g * (ez * dvx - ex * dvz); rz += g * (ex * dvy - ey * dvx);
            }
        }
        float* o = out + 4 * i;
        o[0] = (float)div; o[1] = (float)rx; o[2] = (float)ry; o[3] = (float)rz;
    }
}

// Balsara-type switch (reading C34): B = |div v| / (|div v| + |rot v| + 1e-4 c_s / h): 1 in pure compression, 0 in pure shear
double balsara(const float* r18) {
    const double div = std::fabs((double)r18[13]);
    const double rot = std::sqrt((double)r18[14] * r18[14] + (double)r18[15] * r18[15] + (double)r18[16] * r18[16]);
    return div / (div + rot + 1.0e-4 * (double)r18[12] / (double)r18[3]);
}

// ---- force partial sums of the three-loop cycle: force_block with the viscous term scaled by (B_i + B_j) / 2 ----
// records: FORCE3_IN = [xr0 xr1 xr2 h mass rho rho_dh v0 v1 v2 u P cs div_v rot_v0 rot_v1 rot_v2 time_bin] (time_bin as Table 1's
// column p-f lists it; every particle is active, reading C14, so no arithmetic depends on it)
void force3_block(const float* tgt, uint32_t n_t, const float* src, uint32_t n_s, bool self, float* out, double alpha, double beta) {
    for (uint32_t i = 0; i < n_t; ++i) {
        const float* ri = tgt + 18 * i;
        const double hi = ri[3], rhoi = ri[5], rho_dhi = ri[6], Pi = ri[11], ci = ri[12];
        const double Ai = Pi / ((1.0 + hi * rho_dhi / (3.0 * rhoi)) * rhoi * rhoi);
        const double Bi = balsara(ri);
        double ax = 0, ay = 0, az = 0, dudt = 0, vsig = 0;
        for (uint32_t j = 0; j < n_s; ++j) {
            if (self && j == i) continue;
            const float* rj = src + 18 * j;
            const double hj = rj[3], mj = rj[4], rhoj = rj[5], rho_dhj = rj[6], Pj = rj[11], cj = rj[12];
            const double dx = (double)ri[0] - (double)rj[0], dy = (double)ri[1] - (double)rj[1], dz = (double)ri[2] - (double)rj[2];
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double hcut = std::max(2.0 * hi, 2.0 * hj);
            if (r2 > 0.0 && r2 < hcut * hcut) {
                const double r = std::sqrt(r2);
                const double ex = dx / r, ey = dy / r, ez = dz / r;
                const double Aj = Pj / ((1.0 + hj * rho_dhj / (3.0 * rhoj)) * rhoj * rhoj);
                const double Gi = dW_dr(r, hi), Gj = dW_dr(r, hj), Gbar = 0.5 * (Gi + Gj);
                const double vr = ((double)ri[7] - (double)rj[7]) * ex + ((double)ri[8] - (double)rj[8]) * ey + ((double)ri[9] - (double)rj[9]) * ez;
                const double mu = std::min(0.0, vr);
                const double vs = ci + cj - beta * mu;
                const double Pi_visc = 0.5 * (Bi + balsara(rj)) * (-0.5 * alpha * vs * mu / (0.5 * (rhoi + rhoj)));
                const double fr = -mj * (Ai * Gi + Aj * Gj + Pi_visc * Gbar);
                ax += fr * ex; ay += fr * ey; az += fr * ez;
                dudt += mj * (Ai * Gi + 0.5 * Pi_visc * Gbar) * vr;
                vsig = std::max(vsig, vs);
            }
        }
        float* o = out + 5 * i;
        o[0] = (float)ax; o[1] = (float)ay; o[2] = (float)az; o[3] = (float)dudt; o[4] = (float)vsig;
    }
}

// ---- order of the particles inside a cell (reading C26): ascending Morton code of the position inside the cell
// on a 32 x 32 x 32 sub-grid; equal codes keep generator order.  Sub-cell index along d:
// k_d = clamp(floor((x_d - origin_d) / width * 32), 0, 31); code bit 3b+2 = bit b of k_0 (x), 3b+1 of k_1, 3b of k_2.
uint32_t morton_in_cell(const double* x, const double* origin, double width) {
    uint32_t k[3];
    for (int d = 0; d < 3; ++d) {
        double f = std::floor((x[d] - origin[d]) / width * 32.0);
        if (f < 0.0) f = 0.0;
        if (f > 31.0) f = 31.0;
        k[d] = (uint32_t)f;
    }
    uint32_t code = 0;
    for (int b = 0; b < 5; ++b)
        for (int d = 0; d < 3; ++d) code |= ((k[d] >> b) & 1u) << (3 * b + (2 - d));
    return code;
}

// stable sort of idx[lo, hi) by the Morton code inside the cell (origin, width)
void sort_cell_by_morton(const double* x3, std::vector<uint64_t>& idx, uint64_t lo, uint64_t hi, const double* origin, double width) {
    std::stable_sort(idx.begin() + lo, idx.begin() + hi, [&](uint64_t a, uint64_t b) {
        return morton_in_cell(x3 + 3 * a, origin, width) < morton_in_cell(x3 + 3 * b, origin, width);
    });
}

// periodic minimum gap between [oa, oa+wa] and [ob, ob+wb] along one axis; *shift = image shift of b
double axis_gap(double oa, double wa, double ob, double wb, double box, double* shift, double* second_best) {
    double best = 1e300, second = 1e300, best_s = 0;
    for (int k = -1; k <= 1; ++k) {
        const double s = k * box;
        const double g = std::max(0.0, std::max((ob + s) - (oa + wa), oa - (ob + s + wb)));
        if (g < best) { second = best; best = g; best_s = s; }
        else if (g < second) second = g;
    }
    *shift = best_s; *second_best = second;
    return best;
}

}  // namespace

extern "C" {

int orc_set_threads(int n) { g_threads = n < 1 ? 1 : n; return g_threads; }

double orc_w(double q) { return w_of_q(q); }
double orc_dw(double q) { return dw_of_q(q); }
double orc_W(double r, double h) { return W(r, h); }
double orc_dW_dh(double r, double h) { return dW_dh(r, h); }
double orc_dW_dr(double r, double h) { return dW_dr(r, h); }

int orc_record_bytes(const Attr* attrs, int n_attr, uint32_t flags) {
    if (!attrs_valid(attrs, n_attr)) return -1;
    return record_bytes(attrs, n_attr, flags);
}

// ---- cells: uniform periodic grid (C25 row-major cell index, C26 Morton order inside a cell) ----
// x3: n*3 doubles in [0, box).  perm_out[k] = generator index of the k-th particle in cell order.
int orc_cells_build_grid(const double* x3, uint64_t n, uint32_t cpd, double box, uint64_t* perm_out, Cell* cells_out) {
    const uint64_t nc = (uint64_t)cpd * cpd * cpd;
    std::vector<uint32_t> cell_of(n);
    std::vector<uint64_t> count(nc, 0);
    for (uint64_t p = 0; p < n; ++p) {
        uint32_t idx[3];
        for (int d = 0; d < 3; ++d) {
            const double xv = x3[3 * p + d];
            if (!(xv >= 0.0 && xv < box)) return -2;
            int64_t k = (int64_t)std::floor(xv / box * cpd);
            if (k >= (int64_t)cpd) k = cpd - 1;
            idx[d] = (uint32_t)k;
        }
        cell_of[p] = (idx[0] * cpd + idx[1]) * cpd + idx[2];
        ++count[cell_of[p]];
    }
    std::vector<uint64_t> start(nc + 1, 0);
    for (uint64_t c = 0; c < nc; ++c) start[c + 1] = start[c] + count[c];
    std::vector<uint64_t> fill(start.begin(), start.end() - 1), idx(n);
    for (uint64_t p = 0; p < n; ++p) idx[fill[cell_of[p]]++] = p;         // by cell, generator order inside
    const double w = box / cpd;
    for (uint64_t c = 0; c < nc; ++c) {
        Cell& ce = cells_out[c];
        ce.first = start[c]; ce.count = (uint32_t)count[c]; ce.pad = 0; ce.width = w;
        ce.origin[0] = (double)(c / ((uint64_t)cpd * cpd)) * w;
        ce.origin[1] = (double)((c / cpd) % cpd) * w;
        ce.origin[2] = (double)(c % cpd) * w;
        sort_cell_by_morton(x3, idx, start[c], start[c + 1], ce.origin, w);   // C26
    }
    std::copy(idx.begin(), idx.end(), perm_out);
    return 0;
}

// ---- cells: octree (C21): split a node while it holds more than max_per_leaf
// particles and every non-empty child would still be at least as wide as 2*hmax of its own
// particles.  Leaves in depth-first order, child octant code = 4*bx + 2*by + bz; empty leaves
// are dropped; inside a leaf the particles are in Morton order (C26).  Returns the number of leaves (or < 0); cells_out may be NULL to count only.
static void octree_rec(const double* x3, const float* h, std::vector<uint64_t>& idx, uint64_t lo, uint64_t hi,
                       const double origin[3], double width, uint32_t max_per_leaf, uint32_t depth,
                       std::vector<Cell>& leaves, std::vector<uint64_t>& scratch) {
    const uint64_t cnt = hi - lo;
    if (cnt == 0) return;
    bool split = cnt > max_per_leaf && depth < 20;
    uint64_t ccount[8] = {};
    if (split) {
        float chmax[8] = {};
        for (uint64_t k = lo; k < hi; ++k) {
            const uint64_t p = idx[k];
            int oct = 0;
            for (int d = 0; d < 3; ++d) oct = 2 * oct + (x3[3 * p + d] >= origin[d] + 0.5 * width ? 1 : 0);
            ++ccount[oct];
            chmax[oct] = std::max(chmax[oct], h[p]);
        }
        for (int o = 0; o < 8; ++o)
            if (ccount[o] && !(0.5 * width >= 2.0 * (double)chmax[o])) split = false;
    }
    if (!split) {
        Cell ce; ce.first = lo; ce.count = (uint32_t)cnt; ce.pad = 0; ce.width = width;
        for (int d = 0; d < 3; ++d) ce.origin[d] = origin[d];
        leaves.push_back(ce);
        sort_cell_by_morton(x3, idx, lo, hi, origin, width);              // C26
        return;
    }
    uint64_t cstart[9]; cstart[0] = lo;
    for (int o = 0; o < 8; ++o) cstart[o + 1] = cstart[o] + ccount[o];
    uint64_t fill[8];
    for (int o = 0; o < 8; ++o) fill[o] = cstart[o];
    for (uint64_t k = lo; k < hi; ++k) {                      // stable partition by octant
        const uint64_t p = idx[k];
        int oct = 0;
        for (int d = 0; d < 3; ++d) oct = 2 * oct + (x3[3 * p + d] >= origin[d] + 0.5 * width ? 1 : 0);
        scratch[fill[oct]++] = p;
    }
    std::copy(scratch.begin() + lo, scratch.begin() + hi, idx.begin() + lo);
    for (int o = 0; o < 8; ++o) {
        const double co[3] = {origin[0] + ((o >> 2) & 1) * 0.5 * width, origin[1] + ((o >> 1) & 1) * 0.5 * width,
                              origin[2] + (o & 1) * 0.5 * width};
        octree_rec(x3, h, idx, cstart[o], cstart[o + 1], co, 0.5 * width, max_per_leaf, depth + 1, leaves, scratch);
    }
}

int64_t orc_cells_build_octree(const double* x3, const float* h, uint64_t n, uint32_t max_per_leaf, double box,
                               uint64_t* perm_out, Cell* cells_out, uint64_t cells_cap) {
    std::vector<uint64_t> idx(n), scratch(n);
    for (uint64_t p = 0; p < n; ++p) {
        idx[p] = p;
        for (int d = 0; d < 3; ++d) if (!(x3[3 * p + d] >= 0.0 && x3[3 * p + d] < box)) return -2;
    }
    std::vector<Cell> leaves;
    const double o[3] = {0, 0, 0};
    octree_rec(x3, h, idx, 0, n, o, box, max_per_leaf, 0, leaves, scratch);
    if (perm_out) std::copy(idx.begin(), idx.end(), perm_out);
    if (cells_out) {
        if (leaves.size() > cells_cap) return -3;
        std::copy(leaves.begin(), leaves.end(), cells_out);
    }
    return (int64_t)leaves.size();
}

// ---- tasks (reading step 2): one self task per cell in ascending index,
// then pair tasks (ci < cj) sorted by (ci, cj).  (A, B) is a pair task iff the periodic
// minimum box-to-box gap g(A, B) < max(2 hmax_A, 2 hmax_B).  frame_i = origin_ci,
// frame_j = origin_ci - s with s the image shift that brings cj next to ci.
// Returns n_self + n_pair (or < 0: -4 = a second periodic image is also in range);
// tasks_out may be NULL to count only.  Plain O(n_cells^2).
int64_t orc_tasks_build(const Cell* cells, const float* hmax, uint32_t n_cells, double box, Task* tasks_out,
                        uint64_t tasks_cap, uint64_t* n_self_out, uint64_t* n_pair_out) {
    uint64_t n_out = 0;
    for (uint32_t c = 0; c < n_cells; ++c) {
        if (tasks_out) {
            if (n_out >= tasks_cap) return -3;
            Task& t = tasks_out[n_out];
            t.ci = (int32_t)c; t.cj = -1;
            for (int d = 0; d < 3; ++d) { t.frame_i[d] = cells[c].origin[d]; t.frame_j[d] = cells[c].origin[d]; }
        }
        ++n_out;
    }
    const uint64_t n_self = n_out;
    for (uint32_t a = 0; a < n_cells; ++a) {
        for (uint32_t b = a + 1; b < n_cells; ++b) {
            const double cut = std::max(2.0 * (double)hmax[a], 2.0 * (double)hmax[b]);
            double g2 = 0, shift[3]; bool ambiguous = false;
            for (int d = 0; d < 3; ++d) {
                double second;
                const double g = axis_gap(cells[a].origin[d], cells[a].width, cells[b].origin[d], cells[b].width, box, &shift[d], &second);
                g2 += g * g;
                if (second < cut) ambiguous = true;
            }
            if (!(std::sqrt(g2) < cut)) continue;
            if (ambiguous) return -4;
            if (tasks_out) {
                if (n_out >= tasks_cap) return -3;
                Task& t = tasks_out[n_out];
                t.ci = (int32_t)a; t.cj = (int32_t)b;
                for (int d = 0; d < 3; ++d) { t.frame_i[d] = cells[a].origin[d]; t.frame_j[d] = cells[a].origin[d] - shift[d]; }
            }
            ++n_out;
        }
    }
    if (n_self_out) *n_self_out = n_self;
    if (n_pair_out) *n_pair_out = n_out - n_self;
    return (int64_t)n_out;
}

// Buffer layout of tasks [0, n_tasks) for a given record size; off_out has 2*n_tasks entries.
uint64_t orc_block_offsets(const Cell* cells, const Task* tasks, int64_t n_tasks, int rec_bytes, uint64_t* off_out) {
    std::vector<uint64_t> tmp;
    if (!off_out) { tmp.resize(2 * (size_t)n_tasks); off_out = tmp.data(); }
    return block_offsets(cells, tasks, n_tasks, rec_bytes, off_out);
}

// ---- pack (reading step 5) ----
// For every instance and every entry of the attribute set: copy the bytes; X with FLAG_X_REL_F32:
// rec = (float)(x[d] - frame_side[d]).  Pad bytes of `buf` are left untouched.
int orc_pack(const Part* parts, const Cell* cells, const Task* tasks, int64_t n_tasks, const Attr* attrs, int n_attr,
             uint32_t flags, uint8_t* buf, uint64_t buf_bytes) {
    if (!attrs_valid(attrs, n_attr)) return -1;
    const int rec = record_bytes(attrs, n_attr, flags);
    std::vector<uint64_t> off(2 * (size_t)n_tasks);
    if (block_offsets(cells, tasks, n_tasks, rec, off.data()) > buf_bytes) return -3;
#pragma omp parallel for schedule(dynamic, 64) num_threads(g_threads)
    for (int64_t t = 0; t < n_tasks; ++t) {
        for (int side = 0; side < 2; ++side) {
            const int32_t c = side == 0 ? tasks[t].ci : tasks[t].cj;
            if (c < 0) continue;
            const double* frame = side == 0 ? tasks[t].frame_i : tasks[t].frame_j;
            uint8_t* out = buf + off[2 * t + side];
            for (uint32_t k = 0; k < cells[c].count; ++k) {
                Part& p = const_cast<Part&>(parts[cells[c].first + k]);
                for (int e = 0; e < n_attr; ++e) {
                    const Attr& a = attrs[e];
                    for (int comp = a.comp0; comp < a.comp0 + a.ncomp; ++comp) {
                        if (a.field == X) {
                            if (flags & FLAG_X_REL_F32) { const float xr = (float)(p.x[comp] - frame[comp]); std::memcpy(out, &xr, 4); out += 4; }
                            else { std::memcpy(out, &p.x[comp], 8); out += 8; }
                        } else if (a.field == ID) { std::memcpy(out, &p.id, 8); out += 8; }
                        else if (a.field == TIME_BIN) { const uint8_t b[4] = {(uint8_t)p.time_bin, 0, 0, 0}; std::memcpy(out, b, 4); out += 4; }
                        else { std::memcpy(out, f32_member(p, a.field) + comp, 4); out += 4; }
                    }
                }
            }
        }
    }
    return 0;
}

// ---- unpack (reading step 7, C8) ----
// for task ascending, side i then side j, record ascending: REDUCE: += in f32 for the sum fields,
// fmaxf for v_sig, overwrite for anything else; ASSIGN: overwrite everything.  Serial on purpose.
int orc_unpack(Part* parts, const Cell* cells, const Task* tasks, int64_t n_tasks, const Attr* attrs, int n_attr,
               uint32_t flags, const uint8_t* buf, uint64_t buf_bytes, int mode) {
    if (!attrs_valid(attrs, n_attr)) return -1;
    for (int e = 0; e < n_attr; ++e) if (attrs[e].field == X && (flags & FLAG_X_REL_F32)) return -5;   // not invertible
    const int rec = record_bytes(attrs, n_attr, flags);
    std::vector<uint64_t> off(2 * (size_t)n_tasks);
    if (block_offsets(cells, tasks, n_tasks, rec, off.data()) > buf_bytes) return -3;
    for (int64_t t = 0; t < n_tasks; ++t) {
        for (int side = 0; side < 2; ++side) {
            const int32_t c = side == 0 ? tasks[t].ci : tasks[t].cj;
            if (c < 0) continue;
            const uint8_t* in = buf + off[2 * t + side];
            for (uint32_t k = 0; k < cells[c].count; ++k) {
                Part& p = parts[cells[c].first + k];
                for (int e = 0; e < n_attr; ++e) {
                    const Attr& a = attrs[e];
                    for (int comp = a.comp0; comp < a.comp0 + a.ncomp; ++comp) {
                        if (a.field == X) { std::memcpy(&p.x[comp], in, 8); in += 8; }
                        else if (a.field == ID) { std::memcpy(&p.id, in, 8); in += 8; }
                        else if (a.field == TIME_BIN) { p.time_bin = (int8_t)in[0]; in += 4; }
                        else {
                            float val; std::memcpy(&val, in, 4); in += 4;
                            float* dst = f32_member(p, a.field) + comp;
                            const bool is_sum = a.field == RHO || a.field == RHO_DH || a.field == WCOUNT || a.field == WCOUNT_DH ||
                                                a.field == A || a.field == DU_DT || a.field == DIV_V || a.field == ROT_V;
                            if (mode == MODE_REDUCE && is_sum) *dst = *dst + val;
                            else if (mode == MODE_REDUCE && a.field == V_SIG) *dst = std::fmax(*dst, val);
                            else std::memcpy(dst, &val, 4);
                        }
                    }
                }
            }
        }
    }
    return 0;
}

// ---- zero the outputs of the loop about to run (reading step 4) ----
int orc_zero(Part* parts, uint64_t n, const Attr* attrs, int n_attr) {
    if (!attrs_valid(attrs, n_attr)) return -1;
    for (uint64_t p = 0; p < n; ++p)
        for (int e = 0; e < n_attr; ++e) {
            float* m = f32_member(parts[p], attrs[e].field);
            if (!m) return -1;
            for (int comp = attrs[e].comp0; comp < attrs[e].comp0 + attrs[e].ncomp; ++comp) m[comp] = 0.0f;
        }
    return 0;
}

// ---- density loop over tasks (reading step 6) ----
// in: DENSITY_IN blocks (20-byte records), out: DENSITY_OUT blocks (16-byte records), both in the
// buffer layout above.  A pair task produces results for both sides.
int orc_density(const Cell* cells, const Task* tasks, int64_t n_tasks, const uint8_t* in, uint8_t* out) {
    std::vector<uint64_t> off_in(2 * (size_t)n_tasks), off_out(2 * (size_t)n_tasks);
    block_offsets(cells, tasks, n_tasks, 20, off_in.data());
    block_offsets(cells, tasks, n_tasks, 16, off_out.data());
#pragma omp parallel for schedule(dynamic, 16) num_threads(g_threads)
    for (int64_t t = 0; t < n_tasks; ++t) {
        const uint32_t ni = cells[tasks[t].ci].count;
        const float* bi = (const float*)(in + off_in[2 * t]);
        float* oi = (float*)(out + off_out[2 * t]);
        if (tasks[t].cj < 0) { density_block(bi, ni, bi, ni, oi); continue; }
        const uint32_t nj = cells[tasks[t].cj].count;
        const float* bj = (const float*)(in + off_in[2 * t + 1]);
        float* oj = (float*)(out + off_out[2 * t + 1]);
        density_block(bi, ni, bj, nj, oi);
        density_block(bj, nj, bi, ni, oj);
    }
    return 0;
}

// ---- force loop over tasks (reading step 9) ----
// in: FORCE_IN blocks (52-byte records), out: FORCE_OUT blocks (20-byte records).
int orc_force(const Cell* cells, const Task* tasks, int64_t n_tasks, const uint8_t* in, uint8_t* out, double alpha, double beta) {
    std::vector<uint64_t> off_in(2 * (size_t)n_tasks), off_out(2 * (size_t)n_tasks);
    block_offsets(cells, tasks, n_tasks, 52, off_in.data());
    block_offsets(cells, tasks, n_tasks, 20, off_out.data());
#pragma omp parallel for schedule(dynamic, 16) num_threads(g_threads)
    for (int64_t t = 0; t < n_tasks; ++t) {
        const uint32_t ni = cells[tasks[t].ci].count;
        const float* bi = (const float*)(in + off_in[2 * t]);
        float* oi = (float*)(out + off_out[2 * t]);
        if (tasks[t].cj < 0) { force_block(bi, ni, bi, ni, true, oi, alpha, beta); continue; }
        const uint32_t nj = cells[tasks[t].cj].count;
        const float* bj = (const float*)(in + off_in[2 * t + 1]);
        float* oj = (float*)(out + off_out[2 * t + 1]);
        force_block(bi, ni, bj, nj, false, oi, alpha, beta);
        force_block(bj, nj, bi, ni, false, oj, alpha, beta);
    }
    return 0;
}

// ---- test support: compare two buffers of the same tasks block by block (pad bytes are unspecified and skipped).
// Returns -1 if every record byte agrees, else the byte offset of the first difference inside some block.
int64_t orc_compare_blocks(const Cell* cells, const Task* tasks, int64_t n_tasks, int rec_bytes, const uint8_t* a, const uint8_t* b) {
    std::vector<uint64_t> off(2 * (size_t)n_tasks);
    block_offsets(cells, tasks, n_tasks, rec_bytes, off.data());
    int64_t first_bad = -1;
#pragma omp parallel for schedule(dynamic, 256) num_threads(g_threads)
    for (int64_t t = 0; t < n_tasks; ++t) {
        for (int side = 0; side < 2; ++side) {
            const int32_t c = side == 0 ? tasks[t].ci : tasks[t].cj;
            if (c < 0) continue;
            const uint64_t o = off[2 * t + side], nb = (uint64_t)cells[c].count * rec_bytes;
            if (std::memcmp(a + o, b + o, nb) != 0) {
                uint64_t k = 0;
                while (a[o + k] == b[o + k]) ++k;
#pragma omp critical
                if (first_bad < 0 || (int64_t)(o + k) < first_bad) first_bad = (int64_t)(o + k);
            }
        }
    }
    return first_bad;
}

// ---- reading C31 (test support, not a step of the method): v_sig is a maximum, so it jumps when a pair sits exactly on
// the cut-off r = max(2 h_i, 2 h_j) and f32 / f64 arithmetic decide it differently.  flags_out[p] = 1 for every particle
// that has, in some task, a partner with |r - R_cut| < rel * R_cut; those particles are exempt from the v_sig comparison.
// in: FORCE_IN blocks as packed by orc_pack.
int orc_flag_cutoff_pairs(const Cell* cells, const Task* tasks, int64_t n_tasks, const uint8_t* in, double rel, uint8_t* flags_out) {
    std::vector<uint64_t> off_in(2 * (size_t)n_tasks);
    block_offsets(cells, tasks, n_tasks, 52, off_in.data());
#pragma omp parallel for schedule(dynamic, 16) num_threads(g_threads)
    for (int64_t t = 0; t < n_tasks; ++t) {
        const int32_t ci = tasks[t].ci, cj = tasks[t].cj < 0 ? tasks[t].ci : tasks[t].cj;
        const float* bi = (const float*)(in + off_in[2 * t]);
        const float* bj = tasks[t].cj < 0 ? bi : (const float*)(in + off_in[2 * t + 1]);
        for (uint32_t i = 0; i < cells[ci].count; ++i)
            for (uint32_t j = 0; j < cells[cj].count; ++j) {
                const float *ri = bi + 13 * i, *rj = bj + 13 * j;
                const double dx = (double)ri[0] - (double)rj[0], dy = (double)ri[1] - (double)rj[1], dz = (double)ri[2] - (double)rj[2];
                const double r = std::sqrt(dx * dx + dy * dy + dz * dz), cut = std::max(2.0 * (double)ri[3], 2.0 * (double)rj[3]);
                if (std::fabs(r - cut) < rel * cut) {          // benign race: every writer stores 1
                    flags_out[cells[ci].first + i] = 1;
                    flags_out[cells[cj].first + j] = 1;
                }
            }
    }
    return 0;
}

// ---- gradient loop over tasks (reading C34): in GRADIENT_IN blocks (40-byte records), out GRADIENT_OUT blocks (16-byte records)
int orc_gradient(const Cell* cells, const Task* tasks, int64_t n_tasks, const uint8_t* in, uint8_t* out) {
    std::vector<uint64_t> off_in(2 * (size_t)n_tasks), off_out(2 * (size_t)n_tasks);
    block_offsets(cells, tasks, n_tasks, 40, off_in.data());
    block_offsets(cells, tasks, n_tasks, 16, off_out.data());
#pragma omp parallel for schedule(dynamic, 16) num_threads(g_threads)
    for (int64_t t = 0; t < n_tasks; ++t) {
        const uint32_t ni = cells[tasks[t].ci].count;
        const float* bi = (const float*)(in + off_in[2 * t]);
        float* oi = (float*)(out + off_out[2 * t]);
        if (tasks[t].cj < 0) { gradient_block(bi, ni, bi, ni, true, oi); continue; }
        const uint32_t nj = cells[tasks[t].cj].count;
        const float* bj = (const float*)(in + off_in[2 * t + 1]);
        float* oj = (float*)(out + off_out[2 * t + 1]);
        gradient_block(bi, ni, bj, nj, false, oi);
        gradient_block(bj, nj, bi, ni, false, oj);
    }
    return 0;
}

// ---- force loop of the three-loop cycle: in FORCE3_IN blocks (72-byte records), out FORCE_OUT blocks (20-byte records)
int orc_force3(const Cell* cells, const Task* tasks, int64_t n_tasks, const uint8_t* in, uint8_t* out, double alpha, double beta) {
    std::vector<uint64_t> off_in(2 * (size_t)n_tasks), off_out(2 * (size_t)n_tasks);
    block_offsets(cells, tasks, n_tasks, 72, off_in.data());
    block_offsets(cells, tasks, n_tasks, 20, off_out.data());
#pragma omp parallel for schedule(dynamic, 16) num_threads(g_threads)
    for (int64_t t = 0; t < n_tasks; ++t) {
        const uint32_t ni = cells[tasks[t].ci].count;
        const float* bi = (const float*)(in + off_in[2 * t]);
        float* oi = (float*)(out + off_out[2 * t]);
        if (tasks[t].cj < 0) { force3_block(bi, ni, bi, ni, true, oi, alpha, beta); continue; }
        const uint32_t nj = cells[tasks[t].cj].count;
        const float* bj = (const float*)(in + off_in[2 * t + 1]);
        float* oj = (float*)(out + off_out[2 * t + 1]);
        force3_block(bi, ni, bj, nj, false, oi, alpha, beta);
        force3_block(bj, nj, bi, ni, false, oj, alpha, beta);
    }
    return 0;
}

// brute force O(N^2) with minimum image on the ORIGINAL f64 positions: div_v, rot_v (f64) from v, mass, h, rho as stored
int orc_brute_gradient(const Part* parts, uint64_t n, double box, double* out4) {
#pragma omp parallel for schedule(static) num_threads(g_threads)
    for (int64_t i = 0; i < (int64_t)n; ++i) {
        const Part& pi = parts[i];
        const double hi = pi.h;
        double s[4] = {0, 0, 0, 0};
        for (uint64_t j = 0; j < n; ++j) {
            if ((uint64_t)i == j) continue;
            const Part& pj = parts[j];
            double d[3], r2 = 0;
            for (int k = 0; k < 3; ++k) { d[k] = pi.x[k] - pj.x[k]; d[k] -= box * std::round(d[k] / box); r2 += d[k] * d[k]; }
            if (r2 > 0.0 && r2 < 4.0 * hi * hi) {
                const double r = std::sqrt(r2), g = (double)pj.mass / (double)pj.rho * dW_dr(r, hi);
                const double e[3] = {d[0] / r, d[1] / r, d[2] / r};
                const double dv[3] = {(double)pj.v[0] - pi.v[0], (double)pj.v[1] - pi.v[1], (double)pj.v[2] - pi.v[2]};
                s[0] += g * (dv[0] * e[0] + dv[1] * e[1] + dv[2] * e[2]);
                s[1] += g * (e[1] * dv[2] - e[2] * dv[1]); s[2] += g * (e[2] * dv[0] - e[0] * dv[2]); s[3] += g * (e[0] * dv[1] - e[1] * dv[0]);
            }
        }
        for (int k = 0; k < 4; ++k) out4[4 * i + k] = s[k];
    }
    return 0;
}

// ---- ghost (reading step 8, C12): P = (gamma-1) rho u, c_s = sqrt(gamma (gamma-1) u) ----
int orc_ghost(Part* parts, uint64_t n, double gamma) {
    for (uint64_t p = 0; p < n; ++p) {
        const double rho = parts[p].rho, u = parts[p].u;
        parts[p].P = (float)((gamma - 1.0) * rho * u);
        parts[p].cs = (float)std::sqrt(gamma * (gamma - 1.0) * u);
    }
    return 0;
}

// ---- brute force O(N^2) with minimum image on the ORIGINAL f64 positions (pin for the
// whole cells -> tasks -> pack -> loop -> unpack pipeline).  out4: rho rho_dh wcount wcount_dh (f64).
int orc_brute_density(const Part* parts, uint64_t n, double box, double* out4) {
#pragma omp parallel for schedule(static) num_threads(g_threads)
    for (int64_t i = 0; i < (int64_t)n; ++i) {
        const double hi = parts[i].h;
        double s[4] = {0, 0, 0, 0};
        for (uint64_t j = 0; j < n; ++j) {
            double r2 = 0;
            for (int d = 0; d < 3; ++d) { double dd = parts[i].x[d] - parts[j].x[d]; dd -= box * std::round(dd / box); r2 += dd * dd; }
            if (r2 < 4.0 * hi * hi) {
                const double r = std::sqrt(r2), mj = parts[j].mass;
                s[0] += mj * W(r, hi); s[1] += mj * dW_dh(r, hi); s[2] += W(r, hi); s[3] += dW_dh(r, hi);
            }
        }
        for (int k = 0; k < 4; ++k) out4[4 * i + k] = s[k];
    }
    return 0;
}

// out5: a0 a1 a2 du_dt v_sig (f64); reads rho, rho_dh, P, cs, v, h, mass from the particles
// exactly as stored (f32 values promoted).
int orc_brute_force(const Part* parts, uint64_t n, double box, double alpha, double beta, double* out5) {
#pragma omp parallel for schedule(static) num_threads(g_threads)
    for (int64_t i = 0; i < (int64_t)n; ++i) {
        const Part& pi = parts[i];
        const double hi = pi.h, rhoi = pi.rho;
        const double Ai = (double)pi.P / ((1.0 + hi * (double)pi.rho_dh / (3.0 * rhoi)) * rhoi * rhoi);
        double s[5] = {0, 0, 0, 0, 0};
        for (uint64_t j = 0; j < n; ++j) {
            if ((uint64_t)i == j) continue;
            const Part& pj = parts[j];
            double dx[3], r2 = 0;
            for (int d = 0; d < 3; ++d) { dx[d] = pi.x[d] - pj.x[d]; dx[d] -= box * std::round(dx[d] / box); r2 += dx[d] * dx[d]; }
            const double hj = pj.h, hcut = std::max(2.0 * hi, 2.0 * hj);
            if (r2 > 0.0 && r2 < hcut * hcut) {
                const double r = std::sqrt(r2), rhoj = pj.rho, mj = pj.mass;
                const double Aj = (double)pj.P / ((1.0 + hj * (double)pj.rho_dh / (3.0 * rhoj)) * rhoj * rhoj);
                const double Gi = dW_dr(r, hi), Gj = dW_dr(r, hj), Gbar = 0.5 * (Gi + Gj);
                double vr = 0;
                for (int d = 0; d < 3; ++d) vr += ((double)pi.v[d] - (double)pj.v[d]) * dx[d] / r;
                const double mu = std::min(0.0, vr);
                const double vs = (double)pi.cs + (double)pj.cs - beta * mu;
                const double Pv = -0.5 * alpha * vs * mu / (0.5 * (rhoi + rhoj));
                const double fr = -mj * (Ai * Gi + Aj * Gj + Pv * Gbar);
                for (int d = 0; d < 3; ++d) s[d] += fr * dx[d] / r;
                s[3] += mj * (Ai * Gi + 0.5 * Pv * Gbar) * vr;
                s[4] = std::max(s[4], vs);
            }
        }
        for (int k = 0; k < 5; ++k) out5[5 * i + k] = s[k];
    }
    return 0;
}

// ---- the 48-neighbour condition (BASELINE.json:configs[2]; reading C20) ----
// For each particle solve (4/3) pi (2h)^3 wcount(h) = n_target for h (wcount = sum_j W(r_ij, h),
// self included) by Newton with bisection safeguarding on [h_lo, h_hi] = [h0/2, min(2 h0, h_cap)].
// Candidate neighbours are gathered once from a uniform bin grid of bin width >= 2*h_cap.
// Returns the number of particles that did not converge to |f| <= tol.
int64_t orc_iterate_h(const double* x3, uint64_t n, double box, const float* h0, double h_cap, double n_target, double tol,
                      int max_iter, float* h_out) {
    int nb = (int)std::floor(box / (2.0 * h_cap));
    if (nb < 3) return -2;
    if (nb > 256) nb = 256;
    const double bw = box / nb;
    std::vector<uint32_t> bin_of(n);
    std::vector<uint64_t> start((size_t)nb * nb * nb + 1, 0);
    for (uint64_t p = 0; p < n; ++p) {
        int b[3];
        for (int d = 0; d < 3; ++d) { b[d] = (int)std::floor(x3[3 * p + d] / bw); if (b[d] >= nb) b[d] = nb - 1; if (b[d] < 0) b[d] = 0; }
        bin_of[p] = (uint32_t)((b[0] * nb + b[1]) * nb + b[2]);
        ++start[bin_of[p] + 1];
    }
    for (size_t c = 0; c < start.size() - 1; ++c) start[c + 1] += start[c];
    std::vector<uint64_t> order(n), fill(start.begin(), start.end() - 1);
    for (uint64_t p = 0; p < n; ++p) order[fill[bin_of[p]]++] = p;
    int64_t n_bad = 0;
#pragma omp parallel for schedule(dynamic, 256) num_threads(g_threads) reduction(+ : n_bad)
    for (int64_t i = 0; i < (int64_t)n; ++i) {
        std::vector<double> r_list;
        const int bi = bin_of[i] / (nb * nb), bj = (bin_of[i] / nb) % nb, bk = bin_of[i] % nb;
        const double reach = 2.0 * std::min(2.0 * (double)h0[i], h_cap);
        for (int da = -1; da <= 1; ++da) for (int db = -1; db <= 1; ++db) for (int dc = -1; dc <= 1; ++dc) {
            const int ca = (bi + da + nb) % nb, cb = (bj + db + nb) % nb, cc = (bk + dc + nb) % nb;
            const size_t c = ((size_t)ca * nb + cb) * nb + cc;
            for (uint64_t k = start[c]; k < start[c + 1]; ++k) {
                const uint64_t j = order[k];
                double r2 = 0;
                for (int d = 0; d < 3; ++d) { double dd = x3[3 * i + d] - x3[3 * j + d]; dd -= box * std::round(dd / box); r2 += dd * dd; }
                if (r2 < reach * reach) r_list.push_back(std::sqrt(r2));
            }
        }
        auto f_of = [&](double h, double* dfdh) {
            double wc = 0, wc_dh = 0;
            for (double r : r_list) if (r < 2.0 * h) { wc += W(r, h); wc_dh += dW_dh(r, h); }
            const double c = 32.0 / 3.0 * kPi;
            *dfdh = 3.0 * c * h * h * wc + c * h * h * h * wc_dh;
            return c * h * h * h * wc - n_target;
        };
        double lo = 0.5 * (double)h0[i], hi = std::min(2.0 * (double)h0[i], h_cap), h = std::min((double)h0[i], hi), df;
        double f = f_of(h, &df);
        int it = 0;
        for (; it < max_iter && std::fabs(f) > tol; ++it) {
            if (f > 0) hi = h; else lo = h;
            double hn = df > 0 ? h - f / df : 0.5 * (lo + hi);
            if (!(hn > lo && hn < hi)) hn = 0.5 * (lo + hi);
            h = hn;
            f = f_of(h, &df);
        }
        h_out[i] = (float)h;
        if (std::fabs(f) > tol) ++n_bad;
    }
    return n_bad;
}

}  // extern "C"
