// Host side of the C ABI: errors, layouts, attribute sets, the pack/unpack "programs", the particle store
// and the argument checks in front of every launch.  (include/sph_b200.h documents each entry point.)
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>

#include "internal.h"

namespace sph {

static thread_local char g_err[512] = "";

int32_t fail(int32_t code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int field_ncomp(int f) { return (f == SPH_X || f == SPH_V || f == SPH_A || f == SPH_ROT_V) ? 3 : 1; }
int field_elem_bytes(int f) { return f == SPH_X || f == SPH_ID ? 8 : (f == SPH_TIME_BIN ? 1 : 4); }
bool field_is_f32(int f) { return f != SPH_X && f != SPH_ID && f != SPH_TIME_BIN; }
int comp_record_bytes(int f, uint32_t flags) {
    if (f == SPH_X) return (flags & SPH_ATTR_X_REL_F32) ? 4 : 8;
    if (f == SPH_ID) return 8;
    return 4;
}

int32_t attrset_check(const sph_attrset* set, uint32_t* rec_bytes) {
    if (!set) return fail(SPH_ERR_INVALID_ARG, "attribute set is NULL");
    if (set->n == 0 || set->n > SPH_MAX_ATTR) return fail(SPH_ERR_LAYOUT, "attribute set has %u entries (1..%d)", set->n, SPH_MAX_ATTR);
    if (set->flags & ~SPH_ATTR_X_REL_F32) return fail(SPH_ERR_LAYOUT, "unknown attribute-set flags 0x%x", set->flags);
    bool seen[SPH_NFIELDS][3] = {};
    uint32_t bytes = 0;
    for (uint32_t k = 0; k < set->n; ++k) {
        const sph_attr& a = set->ent[k];
        if (a.field >= SPH_NFIELDS) return fail(SPH_ERR_LAYOUT, "entry %u: field %u does not exist", k, a.field);
        if (a.ncomp < 1 || a.comp0 + a.ncomp > field_ncomp(a.field))
            return fail(SPH_ERR_LAYOUT, "entry %u: components [%u, %u) out of range for field %u", k, a.comp0, a.comp0 + a.ncomp, a.field);
        for (uint32_t c = a.comp0; c < (uint32_t)a.comp0 + a.ncomp; ++c) {
            if (seen[a.field][c]) return fail(SPH_ERR_LAYOUT, "field %u component %u is listed twice", a.field, c);
            seen[a.field][c] = true;
        }
        bytes += a.ncomp * comp_record_bytes(a.field, set->flags);
    }
    if (bytes / 4 > (uint32_t)kMaxRecWords) return fail(SPH_ERR_LAYOUT, "record of %u bytes is too long", bytes);
    if (rec_bytes) *rec_bytes = bytes;
    return SPH_OK;
}

// every record word of (layout, set) as a store location, with the groups the split pack loops partition by
int32_t build_pass_words(const sph_layout& layout, const sph_attrset& set, PassProgram* all) {
    uint32_t rec_bytes = 0;
    if (int32_t rc = attrset_check(&set, &rec_bytes)) return rc;
    std::memset(all, 0, sizeof(*all));
    all->rec_words = rec_bytes / 4;
    uint32_t w = 0;
    for (uint32_t k = 0; k < set.n; ++k) {
        const sph_attr& a = set.ent[k];
        const auto& loc = layout.loc[a.field];
        const uint16_t stride = (uint16_t)layout.stride[loc.sub];
        const uint8_t type = a.field == SPH_X ? 0 : (a.field == SPH_ID ? 2 : (a.field == SPH_TIME_BIN ? 3 : 1));
        auto put = [&](uint32_t off, uint8_t kind, uint8_t comp) {
            all->sel[w] = PassWord{off, stride, loc.sub, kind, (uint8_t)w, comp, {loc.sub, (uint8_t)k, type, (uint8_t)(loc.sub * 4 + type)}};
            ++w;
        };
        for (uint32_t c = a.comp0; c < (uint32_t)a.comp0 + a.ncomp; ++c) {
            const uint32_t off = loc.off + c * field_elem_bytes(a.field);
            if (a.field == SPH_X && (set.flags & SPH_ATTR_X_REL_F32)) put(off, W_XREL, (uint8_t)c);
            else if (a.field == SPH_X || a.field == SPH_ID) { put(off, W_COPY, 0); put(off + 4, W_COPY, 0); }
            else if (a.field == SPH_TIME_BIN) put(off, W_TIMEBIN, 0);
            else put(off, W_COPY, 0);
        }
    }
    all->n_sel = w;
    return SPH_OK;
}

// PACK program: which substruct arrays to stage (and which 16-byte pieces of them), the pre-pass, and for every
// record word the staging offset it is copied from.
int32_t build_pack_program(const sph_layout& layout, const sph_attrset& set, Program* prog) {
    uint32_t rec_bytes = 0;
    if (int32_t rc = attrset_check(&set, &rec_bytes)) return rc;
    std::memset(prog, 0, sizeof(*prog));
    prog->rec_words = rec_bytes / 4;
    prog->xw[0] = prog->xw[1] = prog->xw[2] = 0xFFFFFFFFu;
    // 1) record words as (substruct, byte offset, bytes needed there), before staging offsets are known
    struct Raw { uint8_t sub; uint16_t off; uint8_t kind; } raw[kMaxRecWords];
    uint32_t w = 0;
    bool need[SPH_MAX_SUB][4096 / 16] = {};   // 16-byte pieces of each substruct that hold requested bytes
    bool used[SPH_MAX_SUB] = {};
    auto mark = [&](uint8_t sub, uint32_t off, uint32_t nbytes) {
        used[sub] = true;
        for (uint32_t b = off; b < off + nbytes; ++b) need[sub][b / 16] = true;
    };
    for (uint32_t k = 0; k < set.n; ++k) {
        const sph_attr& a = set.ent[k];
        const auto& loc = layout.loc[a.field];
        for (uint32_t c = a.comp0; c < (uint32_t)a.comp0 + a.ncomp; ++c) {
            const uint16_t off = (uint16_t)(loc.off + c * field_elem_bytes(a.field));
            if (a.field == SPH_X && (set.flags & SPH_ATTR_X_REL_F32)) {
                // the pre-pass leaves f32(x[c] - frame[c]) at x + 4c; it reads all three coordinates
                prog->xw[c] = w;
                raw[w++] = Raw{loc.sub, (uint16_t)(loc.off + 4 * c), (uint8_t)W_XREL};
                mark(loc.sub, loc.off, 24);
            } else if (a.field == SPH_X || a.field == SPH_ID) {
                raw[w++] = Raw{loc.sub, off, (uint8_t)W_COPY};
                raw[w++] = Raw{loc.sub, (uint16_t)(off + 4), (uint8_t)W_COPY};
                mark(loc.sub, off, 8);
            } else if (a.field == SPH_TIME_BIN) {
                raw[w++] = Raw{loc.sub, off, (uint8_t)W_TIMEBIN};
                mark(loc.sub, off, 1);
            } else {
                raw[w++] = Raw{loc.sub, off, (uint8_t)W_COPY};
                mark(loc.sub, off, 4);
            }
        }
    }
    // 2) staging layout: every used substruct gets 32 structs' worth of space, particle 0 of a chunk at smem_base
    uint32_t smem = 0, base_of[SPH_MAX_SUB] = {};
    for (uint32_t s = 0; s < layout.n_sub; ++s) {
        if (!used[s]) continue;
        PackSub& su = prog->su[prog->n_sub_used++];
        const uint32_t stride = layout.stride[s];
        su.sub = s;
        su.stride = stride;
        su.gran = stride % 16 == 0 ? 16 : (stride % 8 == 0 ? 8 : 4);
        su.mask = 0xFFFFFFFFu;
        if (su.gran == 16 && stride >= 32 && stride <= 512 && (stride & (stride - 1)) == 0) {
            su.mask = 0;
            for (uint32_t c = 0; c < stride / 16; ++c) if (need[s][c]) su.mask |= 1u << c;
        }
        su.smem_base = base_of[s] = smem;
        smem += (32 * stride + 15) & ~15u;
    }
    // 3) words -> staging offsets; pre-pass parameters
    for (uint32_t k = 0; k < prog->rec_words; ++k) {
        WordDesc& wd = prog->word[k];
        wd.sub = raw[k].sub;
        wd.kind = raw[k].kind;
        wd.stride = (uint16_t)layout.stride[raw[k].sub];
        wd.a = base_of[raw[k].sub] + raw[k].off;
        if (raw[k].kind == W_XREL) {
            prog->xrel = 1;
            prog->x_src = base_of[raw[k].sub] + layout.loc[SPH_X].off;
            prog->x_stride = layout.stride[raw[k].sub];
        } else if (raw[k].kind == W_TIMEBIN) {
            prog->tb = 1;
            prog->tb_src = wd.a;
            prog->tb_stride = wd.stride;
            prog->tb_dst = smem;
            wd.a = smem;
            wd.stride = 4;
            smem += 128;
        }
    }
    prog->smem_per_warp = (smem + 15) & ~15u;
    return SPH_OK;
}

int32_t build_unpack_program(const sph_layout& layout, const sph_attrset& set, int32_t mode, Program* prog) {
    uint32_t rec_bytes = 0;
    if (int32_t rc = attrset_check(&set, &rec_bytes)) return rc;
    if (mode != SPH_UNPACK_REDUCE && mode != SPH_UNPACK_ASSIGN && mode != SPH_UNPACK_REDUCE_ZERO) return fail(SPH_ERR_INVALID_ARG, "unknown unpack mode %d", mode);
    std::memset(prog, 0, sizeof(*prog));
    prog->rec_words = rec_bytes / 4;
    uint32_t w = 0;
    for (uint32_t k = 0; k < set.n; ++k) {
        const sph_attr& a = set.ent[k];
        const auto& loc = layout.loc[a.field];
        const uint16_t stride = (uint16_t)layout.stride[loc.sub];
        if (a.field == SPH_X && (set.flags & SPH_ATTR_X_REL_F32))
            return fail(SPH_ERR_UNSUPPORTED, "X packed as relative f32 cannot be unpacked (the frame shift is not invertible in f32)");
        const bool is_sum = a.field == SPH_RHO || a.field == SPH_RHO_DH || a.field == SPH_WCOUNT || a.field == SPH_WCOUNT_DH ||
                            a.field == SPH_A || a.field == SPH_DU_DT || a.field == SPH_DIV_V || a.field == SPH_ROT_V;
        for (uint32_t c = a.comp0; c < (uint32_t)a.comp0 + a.ncomp; ++c) {
            const uint32_t off = loc.off + c * field_elem_bytes(a.field);
            if (a.field == SPH_X || a.field == SPH_ID) {
                prog->word[w++] = WordDesc{off, stride, loc.sub, (uint8_t)W_ASSIGN};
                prog->word[w++] = WordDesc{off + 4, stride, loc.sub, (uint8_t)W_ASSIGN};
            } else if (a.field == SPH_TIME_BIN) {
                prog->word[w++] = WordDesc{off, stride, loc.sub, (uint8_t)W_ASSIGN_BYTE};
            } else {
                uint8_t kind = W_ASSIGN;
                if (mode != SPH_UNPACK_ASSIGN && is_sum) kind = W_SUM;
                if (mode != SPH_UNPACK_ASSIGN && a.field == SPH_V_SIG) kind = W_MAX;
                prog->word[w++] = WordDesc{off, stride, loc.sub, kind};
            }
        }
    }
    for (uint32_t k = 0; k + 3 < prog->rec_words; ++k) {
        const WordDesc& a = prog->word[k];
        bool ok = a.stride % 16 == 0 && a.a % 16 == 0;
        for (uint32_t j = 0; j < 4 && ok; ++j) {
            const WordDesc& b = prog->word[k + j];
            ok = b.sub == a.sub && b.a == a.a + 4 * j && b.kind != W_ASSIGN_BYTE;
        }
        prog->vec4[k] = ok;
    }
    return SPH_OK;
}

static int32_t store_check(const sph_store* s) {
    if (!s) return fail(SPH_ERR_INVALID_ARG, "store is NULL");
    return SPH_OK;
}

}  // namespace sph

using namespace sph;

extern "C" {

int32_t sph_last_error(char* msg, size_t cap) {
    if (!msg || cap == 0) return SPH_ERR_INVALID_ARG;
    std::snprintf(msg, cap, "%s", g_err);
    return SPH_OK;
}

// ------------------------------------------------------------------ layouts

static void set_loc(sph_layout* l, int field, uint8_t sub, uint16_t off) { l->loc[field].sub = sub; l->loc[field].pad = 0; l->loc[field].off = off; }

int32_t sph_layout_aos(sph_layout* out) {
    if (!out) return fail(SPH_ERR_INVALID_ARG, "out is NULL");
    std::memset(out, 0, sizeof(*out));
    out->n_sub = 1;
    out->stride[0] = SPH_AOS_BYTES;
    static const uint16_t off[SPH_NFIELDS] = {0, 24, 36, 48, 52, 56, 60, 64, 68, 72, 76, 80, 84, 96, 100, 104, 112, 120};
    for (int f = 0; f < SPH_NFIELDS; ++f) set_loc(out, f, 0, off[f]);
    return SPH_OK;
}

int32_t sph_layout_split(sph_layout* out) {
    if (!out) return fail(SPH_ERR_INVALID_ARG, "out is NULL");
    std::memset(out, 0, sizeof(*out));
    out->n_sub = 6;
    const uint32_t stride[6] = {32, 16, 24, 20, 16, 16};
    for (int s = 0; s < 6; ++s) out->stride[s] = stride[s];
    set_loc(out, SPH_X, 0, 0);       set_loc(out, SPH_H, 0, 24);        set_loc(out, SPH_MASS, 0, 28);
    set_loc(out, SPH_RHO, 1, 0);     set_loc(out, SPH_RHO_DH, 1, 4);    set_loc(out, SPH_WCOUNT, 1, 8);  set_loc(out, SPH_WCOUNT_DH, 1, 12);
    set_loc(out, SPH_V, 2, 0);       set_loc(out, SPH_U, 2, 12);        set_loc(out, SPH_P, 2, 16);      set_loc(out, SPH_CS, 2, 20);
    set_loc(out, SPH_A, 3, 0);       set_loc(out, SPH_DU_DT, 3, 12);    set_loc(out, SPH_V_SIG, 3, 16);
    set_loc(out, SPH_ID, 4, 0);      set_loc(out, SPH_TIME_BIN, 4, 8);
    set_loc(out, SPH_DIV_V, 5, 0);   set_loc(out, SPH_ROT_V, 5, 4);
    return SPH_OK;
}

int32_t sph_layout_from_groups(const uint8_t* fields, uint32_t n_fields, const uint32_t* group_sizes, uint32_t n_groups,
                               const uint32_t* min_stride, sph_layout* out) {
    if (!fields || !group_sizes || !out) return fail(SPH_ERR_INVALID_ARG, "NULL argument");
    if (n_fields != SPH_NFIELDS) return fail(SPH_ERR_LAYOUT, "%u fields listed, every one of the %d must appear once", n_fields, SPH_NFIELDS);
    if (n_groups < 1 || n_groups > SPH_MAX_SUB) return fail(SPH_ERR_LAYOUT, "n_groups = %u (1..%d)", n_groups, SPH_MAX_SUB);
    bool seen[SPH_NFIELDS] = {};
    std::memset(out, 0, sizeof(*out));
    out->n_sub = n_groups;
    uint32_t k = 0;
    for (uint32_t g = 0; g < n_groups; ++g) {
        uint32_t off = 0, max_align = 4;
        if (group_sizes[g] == 0) return fail(SPH_ERR_LAYOUT, "group %u is empty", g);
        for (uint32_t i = 0; i < group_sizes[g]; ++i, ++k) {
            if (k >= n_fields) return fail(SPH_ERR_LAYOUT, "group sizes exceed the field list");
            const int f = fields[k];
            if (f >= SPH_NFIELDS || seen[f]) return fail(SPH_ERR_LAYOUT, "field %d is unknown or listed twice", f);
            seen[f] = true;
            const uint32_t eb = field_elem_bytes(f), align = f == SPH_TIME_BIN ? 1 : (eb == 8 ? 8 : 4);
            off = (off + align - 1) / align * align;
            set_loc(out, f, g, off);
            off += eb * field_ncomp(f);
            max_align = std::max(max_align, align);
        }
        uint32_t stride = (off + max_align - 1) / max_align * max_align;
        if (min_stride && min_stride[g] > stride) stride = (min_stride[g] + max_align - 1) / max_align * max_align;
        out->stride[g] = stride;
    }
    if (k != n_fields) return fail(SPH_ERR_LAYOUT, "group sizes cover %u of %u fields", k, n_fields);
    return sph_layout_validate(out);
}

int32_t sph_layout_validate(const sph_layout* l) {
    if (!l) return fail(SPH_ERR_INVALID_ARG, "layout is NULL");
    SPH_API_BEGIN
    if (l->n_sub < 1 || l->n_sub > SPH_MAX_SUB) return fail(SPH_ERR_LAYOUT, "n_sub = %u (1..%d)", l->n_sub, SPH_MAX_SUB);
    std::vector<std::vector<uint8_t>> used(l->n_sub);
    for (uint32_t s = 0; s < l->n_sub; ++s) {
        if (l->stride[s] == 0 || l->stride[s] % 4 != 0 || l->stride[s] > 4096) return fail(SPH_ERR_LAYOUT, "substruct %u: stride %u", s, l->stride[s]);
        used[s].assign(l->stride[s], 0);
    }
    for (int f = 0; f < SPH_NFIELDS; ++f) {
        const auto& loc = l->loc[f];
        if (loc.sub >= l->n_sub) return fail(SPH_ERR_LAYOUT, "field %d: substruct %u does not exist", f, loc.sub);
        const uint32_t eb = field_elem_bytes(f), nb = eb * field_ncomp(f);
        const uint32_t align = f == SPH_TIME_BIN ? 1 : (eb == 8 ? 8 : 4);
        if (loc.off % align) return fail(SPH_ERR_LAYOUT, "field %d: offset %u is not %u-byte aligned", f, loc.off, align);
        if (eb == 8 && l->stride[loc.sub] % 8) return fail(SPH_ERR_LAYOUT, "field %d: 8-byte member in a substruct of stride %u", f, l->stride[loc.sub]);
        if (loc.off + nb > l->stride[loc.sub]) return fail(SPH_ERR_LAYOUT, "field %d: [%u, %u) exceeds stride %u", f, loc.off, loc.off + nb, l->stride[loc.sub]);
        for (uint32_t b = loc.off; b < loc.off + nb; ++b) {
            if (used[loc.sub][b]) return fail(SPH_ERR_LAYOUT, "field %d overlaps another field at substruct %u byte %u", f, loc.sub, b);
            used[loc.sub][b] = 1;
        }
    }
    return SPH_OK;
    SPH_API_END
}

// ------------------------------------------------------------------ attribute sets

int32_t sph_attrset_canonical(int32_t which, sph_attrset* out) {
    if (!out) return fail(SPH_ERR_INVALID_ARG, "out is NULL");
    std::memset(out, 0, sizeof(*out));
    auto add = [&](int field) { out->ent[out->n++] = sph_attr{(uint8_t)field, 0, (uint8_t)field_ncomp(field), 0}; };
    switch (which) {
        case SPH_SET_DENSITY_IN: out->flags = SPH_ATTR_X_REL_F32; add(SPH_X); add(SPH_H); add(SPH_MASS); break;
        case SPH_SET_DENSITY_OUT: add(SPH_RHO); add(SPH_RHO_DH); add(SPH_WCOUNT); add(SPH_WCOUNT_DH); break;
        case SPH_SET_FORCE_IN:
            out->flags = SPH_ATTR_X_REL_F32;
            add(SPH_X); add(SPH_H); add(SPH_MASS); add(SPH_RHO); add(SPH_RHO_DH); add(SPH_V); add(SPH_U); add(SPH_P); add(SPH_CS);
            break;
        case SPH_SET_FORCE_OUT: add(SPH_A); add(SPH_DU_DT); add(SPH_V_SIG); break;
        case SPH_SET_GRADIENT_IN:
            out->flags = SPH_ATTR_X_REL_F32;
            add(SPH_X); add(SPH_V); add(SPH_MASS); add(SPH_H); add(SPH_U); add(SPH_RHO);
            break;
        case SPH_SET_GRADIENT_OUT: add(SPH_DIV_V); add(SPH_ROT_V); break;
        case SPH_SET_FORCE3_IN:
            out->flags = SPH_ATTR_X_REL_F32;
            add(SPH_X); add(SPH_H); add(SPH_MASS); add(SPH_RHO); add(SPH_RHO_DH); add(SPH_V); add(SPH_U); add(SPH_P); add(SPH_CS);
            add(SPH_DIV_V); add(SPH_ROT_V); add(SPH_TIME_BIN);
            break;
        default: return fail(SPH_ERR_INVALID_ARG, "unknown canonical attribute set %d", which);
    }
    return SPH_OK;
}

int32_t sph_attrset_record_bytes(const sph_attrset* set, uint32_t* bytes_out) {
    if (!bytes_out) return fail(SPH_ERR_INVALID_ARG, "bytes_out is NULL");
    return attrset_check(set, bytes_out);
}

// ------------------------------------------------------------------ store

int32_t sph_store_sub_bytes(const sph_layout* layout, uint64_t n, uint32_t sub, uint64_t* bytes_out) {
    if (!layout || !bytes_out) return fail(SPH_ERR_INVALID_ARG, "NULL argument");
    if (sub >= layout->n_sub) return fail(SPH_ERR_RANGE, "substruct %u of %u", sub, layout->n_sub);
    *bytes_out = ((n * layout->stride[sub] + kTailBytes + 255) / 256) * 256;
    return SPH_OK;
}

int32_t sph_store_create(const sph_layout* layout, uint64_t n, int32_t mem_kind, void* const* ext_ptrs, sph_store** out) {
    if (!out) return fail(SPH_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (int32_t rc = sph_layout_validate(layout)) return rc;
    if (mem_kind != SPH_MEM_DEVICE && mem_kind != SPH_MEM_HOST_PINNED) return fail(SPH_ERR_INVALID_ARG, "mem_kind %d", mem_kind);
    if (n == 0 || n >= (1ull << 32) - 64) return fail(SPH_ERR_RANGE, "n = %llu particles (1 .. 2^32-65)", (unsigned long long)n);
    sph_store* s = new (std::nothrow) sph_store();
    if (!s) return fail(SPH_ERR_ALLOC, "host allocation failed");
    s->layout = *layout;
    s->n = n;
    s->mem_kind = mem_kind;
    for (uint32_t k = 0; k < layout->n_sub; ++k) {
        sph_store_sub_bytes(layout, n, k, &s->bytes[k]);
        if (ext_ptrs) {
            if (!ext_ptrs[k] || ((uintptr_t)ext_ptrs[k] & 255)) { delete s; return fail(SPH_ERR_INVALID_ARG, "ext_ptrs[%u] is NULL or not 256-byte aligned", k); }
            s->base[k] = (char*)ext_ptrs[k];
        } else {
            cudaError_t e = mem_kind == SPH_MEM_DEVICE ? cudaMalloc((void**)&s->base[k], s->bytes[k])
                                                       : cudaHostAlloc((void**)&s->base[k], s->bytes[k], cudaHostAllocMapped | cudaHostAllocPortable);
            if (e != cudaSuccess) {
                sph_store_destroy(s);
                return fail(e == cudaErrorMemoryAllocation ? SPH_ERR_ALLOC : SPH_ERR_CUDA, "store allocation of %llu bytes: %s",
                            (unsigned long long)s->bytes[k], cudaGetErrorString(e));
            }
            s->owned[k] = true;
            e = mem_kind == SPH_MEM_DEVICE ? cudaMemset(s->base[k], 0, s->bytes[k]) : (std::memset(s->base[k], 0, s->bytes[k]), cudaSuccess);
            if (e != cudaSuccess) { sph_store_destroy(s); return fail(SPH_ERR_CUDA, "cudaMemset: %s", cudaGetErrorString(e)); }
        }
    }
    *out = s;
    return SPH_OK;
}

int32_t sph_store_destroy(sph_store* s) {
    if (!s) return SPH_OK;
    for (uint32_t k = 0; k < SPH_MAX_SUB; ++k)
        if (s->owned[k] && s->base[k]) { if (s->mem_kind == SPH_MEM_DEVICE) cudaFree(s->base[k]); else cudaFreeHost(s->base[k]); }
    delete s;
    return SPH_OK;
}

int32_t sph_store_sub_ptr(const sph_store* s, uint32_t sub, void** ptr_out) {
    if (int32_t rc = store_check(s)) return rc;
    if (!ptr_out) return fail(SPH_ERR_INVALID_ARG, "ptr_out is NULL");
    if (sub >= s->layout.n_sub) return fail(SPH_ERR_RANGE, "substruct %u of %u", sub, s->layout.n_sub);
    *ptr_out = s->base[sub];
    return SPH_OK;
}

static int32_t sub_copy_check(const sph_store* s, uint32_t sub, const void* host, uint64_t bytes) {
    if (int32_t rc = store_check(s)) return rc;
    if (!host) return fail(SPH_ERR_INVALID_ARG, "host pointer is NULL");
    if (sub >= s->layout.n_sub) return fail(SPH_ERR_RANGE, "substruct %u of %u", sub, s->layout.n_sub);
    if (bytes != s->n * s->layout.stride[sub])
        return fail(SPH_ERR_RANGE, "%llu bytes given, substruct %u holds %llu", (unsigned long long)bytes, sub, (unsigned long long)(s->n * s->layout.stride[sub]));
    return SPH_OK;
}

int32_t sph_store_upload_sub(sph_store* s, uint32_t sub, const void* host_src, uint64_t bytes, void* stream) {
    if (int32_t rc = sub_copy_check(s, sub, host_src, bytes)) return rc;
    SPH_CUDA_TRY(cudaMemcpyAsync(s->base[sub], host_src, bytes, cudaMemcpyDefault, (cudaStream_t)stream));
    return SPH_OK;
}

int32_t sph_store_download_sub(const sph_store* s, uint32_t sub, void* host_dst, uint64_t bytes, void* stream) {
    if (int32_t rc = sub_copy_check(s, sub, host_dst, bytes)) return rc;
    SPH_CUDA_TRY(cudaMemcpyAsync(host_dst, s->base[sub], bytes, cudaMemcpyDefault, (cudaStream_t)stream));
    return SPH_OK;
}

static int32_t range_copy_check(const sph_store* s, uint32_t sub, const void* host, uint64_t first, uint64_t count) {
    if (int32_t rc = store_check(s)) return rc;
    if (!host) return fail(SPH_ERR_INVALID_ARG, "host pointer is NULL");
    if (sub >= s->layout.n_sub) return fail(SPH_ERR_RANGE, "substruct %u of %u", sub, s->layout.n_sub);
    if (first > s->n || count > s->n - first)
        return fail(SPH_ERR_RANGE, "particles [%llu, +%llu) exceed the store (%llu)", (unsigned long long)first, (unsigned long long)count, (unsigned long long)s->n);
    return SPH_OK;
}

int32_t sph_store_upload_range(sph_store* s, uint32_t sub, const void* host_base, uint64_t first, uint64_t count, void* stream) {
    if (int32_t rc = range_copy_check(s, sub, host_base, first, count)) return rc;
    if (count == 0) return SPH_OK;
    const uint64_t st = s->layout.stride[sub];
    SPH_CUDA_TRY(cudaMemcpyAsync(s->base[sub] + first * st, (const char*)host_base + first * st, count * st, cudaMemcpyDefault, (cudaStream_t)stream));
    return SPH_OK;
}

int32_t sph_store_download_range(const sph_store* s, uint32_t sub, void* host_base, uint64_t first, uint64_t count, void* stream) {
    if (int32_t rc = range_copy_check(s, sub, host_base, first, count)) return rc;
    if (count == 0) return SPH_OK;
    const uint64_t st = s->layout.stride[sub];
    SPH_CUDA_TRY(cudaMemcpyAsync((char*)host_base + first * st, s->base[sub] + first * st, count * st, cudaMemcpyDefault, (cudaStream_t)stream));
    return SPH_OK;
}

// host-side (de)interleave between the canonical AoS record and one substruct array
static void transform(const sph_layout& aos, const sph_layout& lay, uint32_t sub, const char* src_aos, char* sub_buf, uint64_t n, bool to_sub) {
    for (int f = 0; f < SPH_NFIELDS; ++f) {
        if (lay.loc[f].sub != sub) continue;
        const uint32_t nb = field_elem_bytes(f) * field_ncomp(f), so = aos.loc[f].off, dof = lay.loc[f].off, st = lay.stride[sub];
        if (to_sub) for (uint64_t p = 0; p < n; ++p) std::memcpy(sub_buf + p * st + dof, src_aos + p * SPH_AOS_BYTES + so, nb);
        else        for (uint64_t p = 0; p < n; ++p) std::memcpy(const_cast<char*>(src_aos) + p * SPH_AOS_BYTES + so, sub_buf + p * st + dof, nb);
    }
}

int32_t sph_store_import_aos(sph_store* s, const void* host_aos, uint64_t n) {
    if (int32_t rc = store_check(s)) return rc;
    if (!host_aos) return fail(SPH_ERR_INVALID_ARG, "host_aos is NULL");
    if (n != s->n) return fail(SPH_ERR_RANGE, "n = %llu but the store holds %llu", (unsigned long long)n, (unsigned long long)s->n);
    sph_layout aos;
    sph_layout_aos(&aos);
    SPH_CUDA_TRY(cudaDeviceSynchronize());
    for (uint32_t k = 0; k < s->layout.n_sub; ++k) {
        const uint64_t nb = n * s->layout.stride[k];
        if (s->mem_kind == SPH_MEM_HOST_PINNED) {
            std::memset(s->base[k], 0, nb);
            transform(aos, s->layout, k, (const char*)host_aos, s->base[k], n, true);
        } else {
            std::vector<char> tmp;
            try { tmp.assign(nb, 0); } catch (...) { return fail(SPH_ERR_ALLOC, "host staging of %llu bytes", (unsigned long long)nb); }
            transform(aos, s->layout, k, (const char*)host_aos, tmp.data(), n, true);
            SPH_CUDA_TRY(cudaMemcpy(s->base[k], tmp.data(), nb, cudaMemcpyHostToDevice));
        }
    }
    return SPH_OK;
}

int32_t sph_store_export_aos(const sph_store* s, void* host_aos, uint64_t n) {
    if (int32_t rc = store_check(s)) return rc;
    if (!host_aos) return fail(SPH_ERR_INVALID_ARG, "host_aos is NULL");
    if (n != s->n) return fail(SPH_ERR_RANGE, "n = %llu but the store holds %llu", (unsigned long long)n, (unsigned long long)s->n);
    sph_layout aos;
    sph_layout_aos(&aos);
    SPH_CUDA_TRY(cudaDeviceSynchronize());
    std::memset(host_aos, 0, n * SPH_AOS_BYTES);
    for (uint32_t k = 0; k < s->layout.n_sub; ++k) {
        const uint64_t nb = n * s->layout.stride[k];
        if (s->mem_kind == SPH_MEM_HOST_PINNED) {
            transform(aos, s->layout, k, (const char*)host_aos, s->base[k], n, false);
        } else {
            std::vector<char> tmp;
            try { tmp.resize(nb); } catch (...) { return fail(SPH_ERR_ALLOC, "host staging of %llu bytes", (unsigned long long)nb); }
            SPH_CUDA_TRY(cudaMemcpy(tmp.data(), s->base[k], nb, cudaMemcpyDeviceToHost));
            transform(aos, s->layout, k, (const char*)host_aos, tmp.data(), n, false);
        }
    }
    return SPH_OK;
}

int32_t sph_store_set_cells(sph_store* s, const sph_cell* cells, uint32_t n_cells) {
    if (int32_t rc = store_check(s)) return rc;
    if (!cells || n_cells == 0) return fail(SPH_ERR_INVALID_ARG, "no cells");
    SPH_API_BEGIN
    std::vector<std::pair<uint64_t, uint64_t>> ranges;
    ranges.reserve(n_cells);
    uint64_t hash = 0xCBF29CE484222325ull ^ n_cells;        // FNV-1a over the (first, count) pairs
    for (uint32_t c = 0; c < n_cells; ++c) {
        if (cells[c].first > s->n || cells[c].count > s->n - cells[c].first)
            return fail(SPH_ERR_RANGE, "cell %u: [%llu, +%u) exceeds the store (%llu)", c,
                        (unsigned long long)cells[c].first, cells[c].count, (unsigned long long)s->n);
        if (cells[c].count) ranges.emplace_back(cells[c].first, cells[c].first + cells[c].count);
        hash = (hash ^ cells[c].first) * 0x100000001B3ull;
        hash = (hash ^ cells[c].count) * 0x100000001B3ull;
    }
    std::sort(ranges.begin(), ranges.end());
    for (size_t k = 1; k < ranges.size(); ++k)
        if (ranges[k].first < ranges[k - 1].second) return fail(SPH_ERR_RANGE, "cell ranges overlap at particle %llu", (unsigned long long)ranges[k].first);
    s->cells.assign(cells, cells + n_cells);
    s->cells_hash = hash;
    return SPH_OK;
    SPH_API_END
}

// ------------------------------------------------------------------ hot path entry points

int32_t sph_store_zero(sph_store* s, const sph_attrset* set, void* stream) {
    if (int32_t rc = store_check(s)) return rc;
    uint32_t rb;
    if (int32_t rc = attrset_check(set, &rb)) return rc;
    for (uint32_t k = 0; k < set->n; ++k)
        if (!field_is_f32(set->ent[k].field)) return fail(SPH_ERR_UNSUPPORTED, "sph_store_zero handles f32 fields only (field %u)", set->ent[k].field);
    Program prog;
    if (int32_t rc = build_unpack_program(s->layout, *set, SPH_UNPACK_ASSIGN, &prog)) return rc;
    return launch_zero(s->view(), s->n, prog, (cudaStream_t)stream);
}

// cells [cell_first, +cell_count) of the store's table -> the batch's cell chunks [cc0, cc0 + ncc)
static int32_t cell_range(const sph_batch* b, uint32_t cell_first, uint32_t cell_count, uint32_t* cc0, uint32_t* ncc) {
    const uint32_t n_cells = (uint32_t)b->cell_chunk0.size() - 1;
    if (cell_first > n_cells || cell_count > n_cells - cell_first)
        return fail(SPH_ERR_RANGE, "cells [%u, +%u) exceed the cell table (%u)", cell_first, cell_count, n_cells);
    *cc0 = b->cell_chunk0[cell_first];
    *ncc = b->cell_chunk0[cell_first + cell_count] - *cc0;
    return SPH_OK;
}

// A batch indexes particles through the cell table it was built against: it may be used with any store that holds the
// same number of particles under the same cell table (e.g. an AoS and a split-AoS store of one particle set).
static int32_t batch_store_check(const sph_store* s, const sph_batch* b) {
    if (b->store_n != s->n) return fail(SPH_ERR_INVALID_ARG, "batch was built for a store of %llu particles", (unsigned long long)b->store_n);
    if (b->cells_hash != s->cells_hash) return fail(SPH_ERR_INVALID_ARG, "batch was built against another cell table than the store's");
    return SPH_OK;
}

static int32_t transfer_check(const sph_store* s, const sph_batch* b, const sph_attrset* set, const void* d_buf) {
    if (int32_t rc = store_check(s)) return rc;
    if (!b || !d_buf) return fail(SPH_ERR_INVALID_ARG, "batch or buffer is NULL");
    if (!set) return fail(SPH_ERR_INVALID_ARG, "attribute set is NULL");
    return batch_store_check(s, b);
}

int32_t sph_pack_cells(const sph_store* s, const sph_batch* b, const sph_attrset* set, void* d_buf, uint64_t buf_bytes,
                       uint32_t cell_first, uint32_t cell_count, void* stream) {
    if (int32_t rc = transfer_check(s, b, set, d_buf)) return rc;
    SPH_API_BEGIN
    Program prog;
    if (int32_t rc = build_pack_program(s->layout, *set, &prog)) return rc;
    const OffsetTable* ot = nullptr;
    if (int32_t rc = ensure_offsets(b, prog.rec_words * 4, &ot)) return rc;
    if (buf_bytes < ot->total) return fail(SPH_ERR_RANGE, "buffer of %llu bytes, %llu needed", (unsigned long long)buf_bytes, (unsigned long long)ot->total);
    if ((uintptr_t)d_buf & 127) return fail(SPH_ERR_INVALID_ARG, "buffer is not 128-byte aligned");
    uint32_t cc0 = 0, ncc = 0;
    if (int32_t rc = cell_range(b, cell_first, cell_count, &cc0, &ncc)) return rc;
    return launch_pack(s->view(), b, prog, ot->d_occ_off128, (char*)d_buf, cc0, ncc, (cudaStream_t)stream);
    SPH_API_END
}

int32_t sph_pack(const sph_store* s, const sph_batch* b, const sph_attrset* set, void* d_buf, uint64_t buf_bytes, void* stream) {
    if (!b) return fail(SPH_ERR_INVALID_ARG, "batch or buffer is NULL");
    return sph_pack_cells(s, b, set, d_buf, buf_bytes, 0, (uint32_t)b->cell_chunk0.size() - 1, stream);
}

int32_t sph_unpack_cells(sph_store* s, const sph_batch* b, const sph_attrset* set, const void* d_buf, uint64_t buf_bytes, int32_t mode,
                         uint32_t cell_first, uint32_t cell_count, void* stream) {
    if (int32_t rc = transfer_check(s, b, set, d_buf)) return rc;
    SPH_API_BEGIN
    Program prog;
    if (int32_t rc = build_unpack_program(s->layout, *set, mode, &prog)) return rc;
    const OffsetTable* ot = nullptr;
    if (int32_t rc = ensure_offsets(b, prog.rec_words * 4, &ot)) return rc;
    if (buf_bytes < ot->total) return fail(SPH_ERR_RANGE, "buffer of %llu bytes, %llu needed", (unsigned long long)buf_bytes, (unsigned long long)ot->total);
    if ((uintptr_t)d_buf & 127) return fail(SPH_ERR_INVALID_ARG, "buffer is not 128-byte aligned");
    uint32_t cc0 = 0, ncc = 0;
    if (int32_t rc = cell_range(b, cell_first, cell_count, &cc0, &ncc)) return rc;
    bool all_assign = true;
    for (uint32_t w = 0; w < prog.rec_words; ++w) all_assign &= prog.word[w].kind == W_ASSIGN || prog.word[w].kind == W_ASSIGN_BYTE;
    return launch_unpack(s->view(), b, prog, ot->d_occ_off128, (const char*)d_buf, all_assign, mode == SPH_UNPACK_REDUCE_ZERO, cc0, ncc, (cudaStream_t)stream);
    SPH_API_END
}

int32_t sph_unpack(sph_store* s, const sph_batch* b, const sph_attrset* set, const void* d_buf, uint64_t buf_bytes, int32_t mode, void* stream) {
    if (!b) return fail(SPH_ERR_INVALID_ARG, "batch or buffer is NULL");
    return sph_unpack_cells(s, b, set, d_buf, buf_bytes, mode, 0, (uint32_t)b->cell_chunk0.size() - 1, stream);
}

static int32_t loop_check(const sph_batch* b, const void* d_in, uint64_t in_bytes, void* d_out, uint64_t out_bytes, uint32_t rec_in,
                          uint32_t rec_out, const OffsetTable** oin, const OffsetTable** oout) {
    if (!b || !d_in || !d_out) return fail(SPH_ERR_INVALID_ARG, "batch or buffer is NULL");
    if (int32_t rc = ensure_offsets(b, rec_in, oin)) return rc;
    if (int32_t rc = ensure_offsets(b, rec_out, oout)) return rc;
    if (in_bytes < (*oin)->total) return fail(SPH_ERR_RANGE, "input buffer of %llu bytes, %llu needed", (unsigned long long)in_bytes, (unsigned long long)(*oin)->total);
    if (out_bytes < (*oout)->total) return fail(SPH_ERR_RANGE, "output buffer of %llu bytes, %llu needed", (unsigned long long)out_bytes, (unsigned long long)(*oout)->total);
    if (((uintptr_t)d_in | (uintptr_t)d_out) & 127) return fail(SPH_ERR_INVALID_ARG, "buffer is not 128-byte aligned");
    return SPH_OK;
}

int32_t sph_density(const sph_batch* b, const void* d_in, uint64_t in_bytes, void* d_out, uint64_t out_bytes, void* stream) {
    SPH_API_BEGIN
    const OffsetTable *oin = nullptr, *oout = nullptr;
    if (int32_t rc = loop_check(b, d_in, in_bytes, d_out, out_bytes, 20, 16, &oin, &oout)) return rc;
    return launch_density(b, (const char*)d_in, (char*)d_out, (cudaStream_t)stream);
    SPH_API_END
}

int32_t sph_force(const sph_batch* b, const void* d_in, uint64_t in_bytes, void* d_out, uint64_t out_bytes, const sph_params* prm, void* stream) {
    if (!prm) return fail(SPH_ERR_INVALID_ARG, "params is NULL");
    SPH_API_BEGIN
    const OffsetTable *oin = nullptr, *oout = nullptr;
    if (int32_t rc = loop_check(b, d_in, in_bytes, d_out, out_bytes, 52, 20, &oin, &oout)) return rc;
    return launch_force(b, (const char*)d_in, (char*)d_out, *prm, (cudaStream_t)stream);
    SPH_API_END
}

int32_t sph_gradient(const sph_batch* b, const void* d_in, uint64_t in_bytes, void* d_out, uint64_t out_bytes, void* stream) {
    SPH_API_BEGIN
    const OffsetTable *oin = nullptr, *oout = nullptr;
    if (int32_t rc = loop_check(b, d_in, in_bytes, d_out, out_bytes, 40, 16, &oin, &oout)) return rc;
    return launch_gradient(b, (const char*)d_in, (char*)d_out, (cudaStream_t)stream);
    SPH_API_END
}

int32_t sph_force3(const sph_batch* b, const void* d_in, uint64_t in_bytes, void* d_out, uint64_t out_bytes, const sph_params* prm, void* stream) {
    if (!prm) return fail(SPH_ERR_INVALID_ARG, "params is NULL");
    SPH_API_BEGIN
    const OffsetTable *oin = nullptr, *oout = nullptr;
    if (int32_t rc = loop_check(b, d_in, in_bytes, d_out, out_bytes, 72, 20, &oin, &oout)) return rc;
    return launch_force3(b, (const char*)d_in, (char*)d_out, *prm, (cudaStream_t)stream);
    SPH_API_END
}

// ---- split pack loops ----

int32_t sph_pack_pass_masks(const sph_layout* layout, const sph_attrset* set, int32_t split, uint64_t* masks_out, uint32_t* n_out) {
    if (!layout || !set || !masks_out || !n_out) return fail(SPH_ERR_INVALID_ARG, "NULL argument");
    if (split < 0 || split > 3) return fail(SPH_ERR_INVALID_ARG, "split must be 0 (by-struct), 1 (by-element), 2 (by-type) or 3 (by-struct-and-type)");
    SPH_API_BEGIN
    if (int32_t rc = sph_layout_validate(layout)) return rc;
    PassProgram all;
    if (int32_t rc = build_pass_words(*layout, *set, &all)) return rc;
    uint32_t n = 0;
    int key_of[kMaxRecWords];
    for (uint32_t w = 0; w < all.n_sel; ++w) {
        const int key = all.sel[w].group[split];
        uint32_t g = 0;
        while (g < n && key_of[g] != key) ++g;
        if (g == n) { key_of[n] = key; masks_out[n++] = 0; }
        masks_out[g] |= 1ull << w;
    }
    *n_out = n;
    return SPH_OK;
    SPH_API_END
}

int32_t sph_pack_pass(const sph_store* s, const sph_batch* b, const sph_attrset* set, uint64_t word_mask, void* d_buf, uint64_t buf_bytes, void* stream) {
    if (int32_t rc = transfer_check(s, b, set, d_buf)) return rc;
    SPH_API_BEGIN
    PassProgram all, pp;
    if (int32_t rc = build_pass_words(s->layout, *set, &all)) return rc;
    if (all.rec_words < 64 && (word_mask >> all.rec_words)) return fail(SPH_ERR_RANGE, "word mask names a word beyond the record's %u", all.rec_words);
    pp = all;
    pp.n_sel = 0;
    for (uint32_t w = 0; w < all.n_sel; ++w)
        if (word_mask >> w & 1) pp.sel[pp.n_sel++] = all.sel[w];
    const OffsetTable* ot = nullptr;
    if (int32_t rc = ensure_offsets(b, all.rec_words * 4, &ot)) return rc;
    if (buf_bytes < ot->total) return fail(SPH_ERR_RANGE, "buffer of %llu bytes, %llu needed", (unsigned long long)buf_bytes, (unsigned long long)ot->total);
    if ((uintptr_t)d_buf & 127) return fail(SPH_ERR_INVALID_ARG, "buffer is not 128-byte aligned");
    return launch_pack_pass(s->view(), pp, b->d_cell_chunks, ot->d_occ_off128, b->d_occ_frames, (char*)d_buf, b->n_cell_chunks, (cudaStream_t)stream);
    SPH_API_END
}

// ---- de-duplicated cell slots ----

int32_t sph_slot_attrset(int32_t loop, sph_attrset* out) {
    if (!out) return fail(SPH_ERR_INVALID_ARG, "out is NULL");
    if (loop < 0 || loop > 1) return fail(SPH_ERR_INVALID_ARG, "loop must be 0 (density) or 1 (force)");
    if (int32_t rc = sph_attrset_canonical(loop == 0 ? SPH_SET_DENSITY_IN : SPH_SET_FORCE_IN, out)) return rc;
    out->flags = 0;                                                                   // x as raw f64: the loop applies the frame
    out->ent[out->n++] = sph_attr{(uint8_t)SPH_TIME_BIN, 0, 1, 0};                    // odd record length (9 / 17 words)
    return SPH_OK;
}

int32_t sph_batch_slot_bytes(const sph_batch* b, int32_t loop, uint64_t* bytes_out) {
    if (!b || !bytes_out) return fail(SPH_ERR_INVALID_ARG, "NULL argument");
    SPH_API_BEGIN
    const SlotTables* sl = nullptr;
    if (int32_t rc = ensure_slots(b, loop, &sl)) return rc;
    *bytes_out = sl->total;
    return SPH_OK;
    SPH_API_END
}

int32_t sph_pack_slots(const sph_store* s, const sph_batch* b, int32_t loop, void* d_slots, uint64_t slot_bytes, void* stream) {
    if (int32_t rc = store_check(s)) return rc;
    if (!b || !d_slots) return fail(SPH_ERR_INVALID_ARG, "batch or buffer is NULL");
    if (int32_t rc = batch_store_check(s, b)) return rc;
    SPH_API_BEGIN
    sph_attrset set;
    if (int32_t rc = sph_slot_attrset(loop, &set)) return rc;
    const SlotTables* sl = nullptr;
    if (int32_t rc = ensure_slots(b, loop, &sl)) return rc;
    Program prog;
    if (int32_t rc = build_pack_program(s->layout, set, &prog)) return rc;
    if (prog.rec_words * 4 != sl->rec_bytes) return fail(SPH_ERR_LAYOUT, "slot record of %u bytes, %u expected", prog.rec_words * 4, sl->rec_bytes);
    if (slot_bytes < sl->total) return fail(SPH_ERR_RANGE, "slot buffer of %llu bytes, %llu needed", (unsigned long long)slot_bytes, (unsigned long long)sl->total);
    if ((uintptr_t)d_slots & 127) return fail(SPH_ERR_INVALID_ARG, "buffer is not 128-byte aligned");
    return launch_pack_tables(s->view(), prog, sl->d_chunks, sl->d_slot_off128, sl->d_zero_frames, (char*)d_slots, sl->n_chunks, (cudaStream_t)stream);
    SPH_API_END
}

static int32_t slot_loop_check(const sph_batch* b, int loop, const void* d_slots, uint64_t slot_bytes, void* d_out, uint64_t out_bytes, const SlotTables** sl) {
    if (!b || !d_slots || !d_out) return fail(SPH_ERR_INVALID_ARG, "batch or buffer is NULL");
    if (int32_t rc = ensure_slots(b, loop, sl)) return rc;
    const OffsetTable* oout = nullptr;
    if (int32_t rc = ensure_offsets(b, loop == 0 ? 16 : 20, &oout)) return rc;
    if (slot_bytes < (*sl)->total) return fail(SPH_ERR_RANGE, "slot buffer of %llu bytes, %llu needed", (unsigned long long)slot_bytes, (unsigned long long)(*sl)->total);
    if (out_bytes < oout->total) return fail(SPH_ERR_RANGE, "output buffer of %llu bytes, %llu needed", (unsigned long long)out_bytes, (unsigned long long)oout->total);
    if (((uintptr_t)d_slots | (uintptr_t)d_out) & 127) return fail(SPH_ERR_INVALID_ARG, "buffer is not 128-byte aligned");
    return SPH_OK;
}

int32_t sph_density_slots(const sph_batch* b, const void* d_slots, uint64_t slot_bytes, void* d_out, uint64_t out_bytes, void* stream) {
    SPH_API_BEGIN
    const SlotTables* sl = nullptr;
    if (int32_t rc = slot_loop_check(b, 0, d_slots, slot_bytes, d_out, out_bytes, &sl)) return rc;
    return launch_density_slots(b, *sl, (const char*)d_slots, (char*)d_out, (cudaStream_t)stream);
    SPH_API_END
}

int32_t sph_force_slots(const sph_batch* b, const void* d_slots, uint64_t slot_bytes, void* d_out, uint64_t out_bytes, const sph_params* prm, void* stream) {
    if (!prm) return fail(SPH_ERR_INVALID_ARG, "params is NULL");
    SPH_API_BEGIN
    const SlotTables* sl = nullptr;
    if (int32_t rc = slot_loop_check(b, 1, d_slots, slot_bytes, d_out, out_bytes, &sl)) return rc;
    return launch_force_slots(b, *sl, (const char*)d_slots, (char*)d_out, *prm, (cudaStream_t)stream);
    SPH_API_END
}

int32_t sph_ghost(sph_store* s, const sph_params* prm, void* stream) {
    if (int32_t rc = store_check(s)) return rc;
    if (!prm) return fail(SPH_ERR_INVALID_ARG, "params is NULL");
    return launch_ghost(s->view(), s->n, s->layout, *prm, (cudaStream_t)stream);
}

}  // extern "C"
