// Internal declarations of libsph_b200 (not part of the C ABI; see include/sph_b200.h).
#pragma once

#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <map>
#include <mutex>
#include <new>
#include <vector>

#include "sph_b200.h"

namespace sph {

int32_t fail(int32_t code, const char* fmt, ...);
// Every extern "C" body that can allocate sits between these two: nothing is thrown across the C ABI.
#define SPH_API_BEGIN try {
#define SPH_API_END                                                                                         \
    }                                                                                                       \
    catch (const std::bad_alloc&) { return ::sph::fail(SPH_ERR_ALLOC, "host allocation failed"); }          \
    catch (...) { return ::sph::fail(SPH_ERR_INVALID_ARG, "unexpected C++ exception"); }
#define SPH_CUDA_TRY(expr)                                                                             \
    do {                                                                                               \
        cudaError_t e_ = (expr);                                                                       \
        if (e_ != cudaSuccess) return ::sph::fail(SPH_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
    } while (0)

// ---- field metadata ----
int field_ncomp(int field);                 // 3 for X, V, A, ROT_V, else 1
int field_elem_bytes(int field);            // bytes of one component in the STORE: X 8, ID 8, TIME_BIN 1, else 4
int comp_record_bytes(int field, uint32_t flags);   // bytes of one component in a RECORD
bool field_is_f32(int field);
int32_t attrset_check(const sph_attrset* set, uint32_t* rec_bytes);

constexpr int kMaxRecWords = 48;   // all 26 scalars + raw x (6 words) + id (2 words) = 33; a little slack
constexpr uint32_t kTailBytes = 64;   // readable slack after every substruct array

// ---- device-side views ----
struct StoreView {
    char* base[SPH_MAX_SUB];
    uint32_t stride[SPH_MAX_SUB];
};

// one block of a buffer = one side of one task
struct SideRec {
    uint32_t first;    // first particle of the cell
    uint32_t count;    // particles in the cell
    uint32_t pad;
    uint32_t cell;
};

// one 32-particle slice of a cell that occurs in the batch (work item of unpack)
struct CellChunk {
    uint32_t first;    // first particle of the slice
    uint32_t count;    // 1..32
    uint32_t k0;       // offset of the slice inside its cell (multiple of 32)
    uint32_t occ0;     // [occ0, occ0 + nocc): the cell's blocks in ascending (task, side) order
    uint32_t nocc;
};

constexpr uint32_t kLoopTargets = 64;
// work item of the density / force loops: up to 64 targets of one block (two per lane) against the block they gather from.  Offsets in units of 128 bytes into the loop's input / output buffer (chunk starts are multiples of 128 bytes).
struct LoopItem {
    uint32_t tin128;     // the targets' input records
    uint32_t sin128;     // first input record of the source block
    uint32_t tout128;    // the targets' result records
    uint32_t nt_ns;      // targets (1..64) | sources << 7
};

// word kinds of the pack / unpack programs
enum : uint32_t { W_COPY = 0, W_XREL = 1, W_TIMEBIN = 2,            // pack (host side only: the kernel sees plain copies)
                  W_SUM = 3, W_MAX = 4, W_ASSIGN = 5, W_ASSIGN_BYTE = 6, W_SKIP = 7 };   // unpack

// Per record word: where it comes from / goes to.  Built on the host from (layout, attribute set).
//   pack:   a = byte offset of the word of particle 0 inside the warp's staging area (after the pre-pass every word
//           is a plain 4-byte copy), stride = bytes between consecutive particles there
//   unpack: a = byte offset inside the substruct, stride = the substruct's stride, sub, kind
struct WordDesc {
    uint32_t a;
    uint16_t stride;
    uint8_t sub;
    uint8_t kind;
};

// One substruct array a pack program draws from, staged per 32-particle chunk with particle 0 at smem_base.
struct PackSub {
    const char* base;     // the substruct array (filled in at launch from the store)
    uint32_t sub;
    uint32_t stride;
    uint32_t gran;        // 16, 8 or 4: the largest power of two that divides the stride (cp.async size)
    uint32_t mask;        // gran == 16 and power-of-two stride in [32, 512]: bit c set = 16-byte piece c of the struct is needed
    uint32_t smem_base;   // 16-byte aligned
};

struct Program {
    uint32_t rec_words;
    uint32_t n_sub_used;
    uint32_t smem_per_warp;        // bytes of staging per warp (pack)
    // pack pre-pass, one lane per particle: x (3 f64 at x_src + k x_stride) -> f32(x - frame) written over its first 12 bytes;
    // time_bin (1 byte at tb_src + k tb_stride) -> zero-extended word at tb_dst + 4k
    uint32_t xrel, x_src, x_stride;
    uint32_t xw[3];                // record word that holds f32(x[c] - frame[c]), or 0xFFFFFFFF
    uint32_t tb, tb_src, tb_stride, tb_dst;
    PackSub su[SPH_MAX_SUB];
    WordDesc word[kMaxRecWords];
    uint8_t vec4[kMaxRecWords];    // unpack: words w..w+3 are 16 contiguous, 16-byte aligned bytes of one substruct (all plain f32 words)
};

// One pass of a split pack loop (PAPER.md:150-152 loop fission): the selected record words only, each read
// straight from the store and written into its place in every record of every block.
struct PassWord {
    uint32_t off;        // byte offset inside the substruct (W_XREL: of the f64 coordinate)
    uint16_t stride;
    uint8_t sub, kind;   // W_COPY, W_XREL, W_TIMEBIN
    uint8_t w, comp;     // record word; W_XREL: which coordinate
    uint8_t group[4];    // substruct, attribute entry, data type (0 f64, 1 f32, 2 i64, 3 i8), substruct x type
};
struct PassProgram {
    uint32_t rec_words, n_sel;
    PassWord sel[kMaxRecWords];
};
int32_t build_pass_words(const sph_layout& layout, const sph_attrset& set, PassProgram* all);      // every record word, in record order
int32_t launch_pack_pass(const StoreView& view, const PassProgram& pp, const CellChunk* d_chunks, const uint32_t* d_occ_off128, const double* d_occ_frames,
                         char* d_buf, uint32_t ncc, cudaStream_t st);

int32_t build_pack_program(const sph_layout& layout, const sph_attrset& set, Program* prog);
int32_t build_unpack_program(const sph_layout& layout, const sph_attrset& set, int32_t mode, Program* prog);

// De-duplicated cell slots ("data replication"): every cell the batch touches is packed once,
// x as raw f64, and the loops' items index slots and carry the frames of their two sides.  One set of tables per loop.
struct SlotTables {
    bool built = false;
    uint32_t rec_bytes = 0;                // 36 (density) or 68 (force)
    uint64_t total = 0;                    // bytes of the slot buffer
    uint32_t n_chunks = 0;
    CellChunk* d_chunks = nullptr;         // 32-particle chunks of the touched cells; every chunk has one occurrence: its cell's slot
    uint32_t* d_slot_off128 = nullptr;     // per touched cell: slot start in units of 128 bytes
    double* d_zero_frames = nullptr;       // 3 zeros per touched cell (the pack kernel subtracts nothing)
    LoopItem* d_items = nullptr;           // the loop's items with tin128 / sin128 pointing into the slot buffer
    double* d_item_frames = nullptr;       // per item: frame of the targets' side (3), frame of the sources' side (3)
};

struct ItemSide { uint32_t tgt, src, kc; };    // a loop item: 64-target chunk kc of block tgt against block src

struct OffsetTable {
    uint32_t* d_off128 = nullptr;          // per side: block start in units of 128 bytes
    uint32_t* d_occ_off128 = nullptr;      // per occurrence (cell-major, ascending side): the same, for the ordered unpack
    std::vector<uint64_t> h_off;           // per side, bytes
    std::vector<uint64_t> seg_off;         // per segment, bytes
    uint64_t total = 0;
};

}  // namespace sph

struct sph_store {
    sph_layout layout;
    uint64_t n = 0;
    int32_t mem_kind = SPH_MEM_DEVICE;
    char* base[SPH_MAX_SUB] = {};
    bool owned[SPH_MAX_SUB] = {};
    uint64_t bytes[SPH_MAX_SUB] = {};
    std::vector<sph_cell> cells;
    uint64_t cells_hash = 0;      // of the (first, count) pairs of the cell table: what a batch is tied to
    sph::StoreView view() const {
        sph::StoreView v{};
        for (uint32_t s = 0; s < layout.n_sub; ++s) { v.base[s] = base[s]; v.stride[s] = layout.stride[s]; }
        return v;
    }
};

struct sph_batch {
    uint64_t n_tasks = 0, n_self = 0, n_pair = 0;
    uint32_t n_sides = 0, n_cell_chunks = 0, n_occ = 0, n_segments = 1, tasks_per_segment = 0, max_count = 0, max_nocc = 0;
    uint64_t n_instances = 0, n_candidates = 0, n_cells_touched = 0, store_n = 0, max_item_candidates = 0;
    uint64_t cells_hash = 0;                  // of the cell table the batch was built against
    std::vector<sph::SideRec> sides;          // host copy
    std::vector<uint32_t> occ_side;           // host copy of the occurrence lists
    std::vector<uint32_t> task_side0;         // n_tasks + 1
    std::vector<uint32_t> cell_chunk0;        // n_cells + 1: first 32-particle cell chunk of every cell of the store's table
    // device tables
    double* d_occ_frames = nullptr;           // 3 per occurrence (cell-major, ascending side): the frame of that side
    sph::CellChunk* d_cell_chunks = nullptr;
    sph::LoopItem* d_items_density = nullptr; // one per 64-target chunk of a block (20-byte in, 16-byte out records)
    sph::LoopItem* d_items_force = nullptr;   // (52-byte in, 20-byte out records)
    sph::LoopItem* d_items_gradient = nullptr;   // three-loop cycle: 40-byte in, 16-byte out records
    sph::LoopItem* d_items_force3 = nullptr;     //                   72-byte in, 20-byte out records
    uint32_t n_items = 0;                     // items are cell-major: the chunks of a cell's occurrences follow one another
    // block offsets by record bytes: the only part that grows after sph_batch_create (a table is built the first time a
    // record size is asked for, under the mutex; tables are never removed, so pointers to them stay valid)
    mutable std::mutex mu;
    mutable std::map<uint32_t, sph::OffsetTable> offsets;
    // cell slots (built the first time a slot call needs them, under the mutex)
    std::vector<sph::ItemSide> item_side;     // the items in launch order
    std::vector<double> side_frames;          // 3 per side
    mutable sph::SlotTables slots[2];         // [0] density, [1] force
};

namespace sph {
int32_t ensure_offsets(const sph_batch* batch, uint32_t rec_bytes, const OffsetTable** out);
int32_t ensure_slots(const sph_batch* batch, int loop, const SlotTables** out);      // loop: 0 density, 1 force
int32_t device_sms(int* sms_out);      // SM count of the current device

// kernel launchers (kernels_*.cu)
// [cc0, cc0 + ncc): the cell chunks to work on
int32_t launch_pack(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_occ_off128, char* d_buf,
                    uint32_t cc0, uint32_t ncc, cudaStream_t st);
int32_t launch_unpack(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_occ_off128, const char* d_buf,
                      bool last_only, bool from_zero, uint32_t cc0, uint32_t ncc, cudaStream_t st);
int32_t launch_density(const sph_batch* b, const char* d_in, char* d_out, cudaStream_t st);
int32_t launch_force(const sph_batch* b, const char* d_in, char* d_out, const sph_params& prm, cudaStream_t st);
int32_t launch_density_slots(const sph_batch* b, const SlotTables& sl, const char* d_slots, char* d_out, cudaStream_t st);
int32_t launch_force_slots(const sph_batch* b, const SlotTables& sl, const char* d_slots, char* d_out, const sph_params& prm, cudaStream_t st);
int32_t launch_pack_tables(const StoreView& view, const Program& prog, const CellChunk* d_chunks, const uint32_t* d_occ_off128, const double* d_occ_frames,
                           char* d_buf, uint32_t ncc, cudaStream_t st);
int32_t launch_gradient(const sph_batch* b, const char* d_in, char* d_out, cudaStream_t st);
int32_t launch_force3(const sph_batch* b, const char* d_in, char* d_out, const sph_params& prm, cudaStream_t st);
int32_t launch_zero(const StoreView& view, uint64_t n, const Program& prog, cudaStream_t st);
int32_t launch_ghost(const StoreView& view, uint64_t n, const sph_layout& layout, const sph_params& prm, cudaStream_t st);
}  // namespace sph
