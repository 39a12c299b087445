// sph_pack_static: PACK for callers that are not allowed to allocate device memory.
//
// Who that is.  The paper's setting is a task-based SPH code whose worker threads each drive their own CUDA stream
// (PAPER.md:80, 98).  Such a host program usually takes all the device memory it will ever use once, at start-up, and
// hands pieces of it to the tasks; from then on no thread may call cudaMalloc / cudaFree, because (a) on a nearly full
// GPU (a 2^26-particle store, BASELINE.json configs[4]) a late allocation can simply fail, and (b) cudaMalloc and cudaFree
// may wait for every stream of the device, so one worker that allocates stalls the packs and loops of all the others.
// The ordinary path (sph_batch_create + sph_pack) does allocate: a batch owns device tables (32-particle cell chunks,
// block offsets, frames) that the pack kernel reads beside the store and the buffer.
//
// What this file does instead.  The same tables are built on the host for the tasks of ONE call, copied into a fixed
// array that is part of the library's device image (g_pack_scratch below, kScratchBytes = 2.1 MiB; every GPU that loads
// libsph_b200.so holds that much until the process ends), and the unchanged pack kernel is launched on them.  The host
// side works in fixed arrays of this file as well, so the call uses no heap either.  It calls no cudaMalloc, cudaFree,
// cudaHostAlloc or any other allocating routine.
//
// The price: the sizes are capped (SPH_PACK_STATIC_MAX_TASKS, SPH_PACK_STATIC_MAX_CHUNKS in sph_b200.h), every call pays
// the table upload again, and all calls share the one array -- see the entry point's comment for what that forbids.
#include <algorithm>
#include <cstring>

#include "internal.h"

using namespace sph;

namespace {

constexpr uint32_t kMaxTasks = SPH_PACK_STATIC_MAX_TASKS;
constexpr uint32_t kMaxSides = 2 * kMaxTasks;                   // a pair task has two sides (blocks)
constexpr uint32_t kMaxChunks = SPH_PACK_STATIC_MAX_CHUNKS;     // 32-particle slices of the cells a call touches
constexpr int kMaxDevices = 64;

// the three tables the pack kernel reads, at fixed places of the scratch array (each a multiple of 256 bytes)
constexpr size_t kChunksAt = 0;                                                   // CellChunk[kMaxChunks]
constexpr size_t kFramesAt = kChunksAt + (size_t)kMaxChunks * sizeof(CellChunk);  // double[kMaxSides][3], cell-major occurrences
constexpr size_t kOffsetsAt = kFramesAt + (size_t)kMaxSides * 3 * sizeof(double); // uint32_t[kMaxSides], block starts / 128
constexpr size_t kScratchBytes = kOffsetsAt + (size_t)kMaxSides * sizeof(uint32_t);
static_assert(kFramesAt % 256 == 0 && kOffsetsAt % 256 == 0, "tables must keep the array's alignment");
static_assert(kScratchBytes <= (4u << 20), "the resident scratch array is meant to stay small");

// The scratch itself: lives in the device image of the library, one copy per GPU.  In HOST code this name is only a
// handle for cudaGetSymbolAddress -- it is not a device address and must never be handed to a kernel or a memcpy as one.
static __device__ __align__(256) unsigned char g_pack_scratch[kScratchBytes];

// host-side state: the device address of g_pack_scratch per device ordinal, and the arrays the tables are built in
std::mutex g_mu;                                  // one call at a time builds and uploads tables
unsigned char* g_scratch_addr[kMaxDevices] = {};  // filled by the first call on each device
alignas(16) unsigned char h_tables[kScratchBytes];   // host image of the three tables (same places as on the device)
uint64_t h_key[kMaxSides];                        // (cell << 32 | side): sorted = the occurrence lists, cell-major
uint32_t h_side_task[kMaxSides];                  // side -> task << 1 | (0: side i, 1: side j)
uint32_t h_side_off128[kMaxSides];                // side -> block start in units of 128 bytes

// once per device, with that device current: where g_pack_scratch lives on it
int32_t scratch_address(unsigned char** out) {
    int dev = -1;
    SPH_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(SPH_ERR_UNSUPPORTED, "device ordinal %d (sph_pack_static keeps %d addresses)", dev, kMaxDevices);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_pack_scratch);
        if (e != cudaSuccess || !p) return fail(SPH_ERR_CUDA, "cudaGetSymbolAddress(g_pack_scratch) on device %d: %s", dev, cudaGetErrorString(e));
        g_scratch_addr[dev] = (unsigned char*)p;
    }
    *out = g_scratch_addr[dev];
    return SPH_OK;
}

}  // namespace

extern "C" int32_t sph_pack_static(const sph_store* s, const sph_task* tasks, uint32_t n_tasks, const sph_attrset* set, void* d_buf,
                                   uint64_t buf_bytes, uint64_t* bytes_needed_out, void* stream) {
    if (bytes_needed_out) *bytes_needed_out = 0;
    if (!s || !tasks || !set) return fail(SPH_ERR_INVALID_ARG, "store, tasks or attribute set is NULL");
    if (!d_buf && !bytes_needed_out) return fail(SPH_ERR_INVALID_ARG, "buffer is NULL (allowed only as a size query, with bytes_needed_out)");
    if (n_tasks == 0) return fail(SPH_ERR_INVALID_ARG, "no tasks");
    if (s->cells.empty()) return fail(SPH_ERR_INVALID_ARG, "the store has no cell table (sph_store_set_cells)");
    if (n_tasks > kMaxTasks)
        return fail(SPH_ERR_RANGE, "sph_pack_static takes at most %u tasks per call (SPH_PACK_STATIC_MAX_TASKS), got %u: split the bundle or use sph_batch_create + sph_pack",
                    kMaxTasks, n_tasks);
    if ((uintptr_t)d_buf & 127) return fail(SPH_ERR_INVALID_ARG, "buffer is not 128-byte aligned");
    SPH_API_BEGIN
    Program prog;
    if (int32_t rc = build_pack_program(s->layout, *set, &prog)) return rc;
    const uint32_t rec_bytes = prog.rec_words * 4;
    const uint32_t n_cells = (uint32_t)s->cells.size();

    std::lock_guard<std::mutex> lock(g_mu);
    // blocks in buffer order (task by task, side i then side j), laid out as a one-segment batch lays them out
    uint32_t n_sides = 0;
    uint64_t run = 0;
    for (uint32_t t = 0; t < n_tasks; ++t) {
        const sph_task& tk = tasks[t];
        if (tk.ci < 0 || (uint32_t)tk.ci >= n_cells || tk.cj < -1 || (tk.cj >= 0 && (uint32_t)tk.cj >= n_cells) || tk.cj == tk.ci)
            return fail(SPH_ERR_RANGE, "task %u references cells (%d, %d); the store has %u", t, tk.ci, tk.cj, n_cells);
        for (uint32_t side = 0; side < (tk.cj >= 0 ? 2u : 1u); ++side) {
            const uint32_t c = (uint32_t)(side == 0 ? tk.ci : tk.cj);
            h_key[n_sides] = (uint64_t)c << 32 | n_sides;
            h_side_task[n_sides] = t << 1 | side;
            h_side_off128[n_sides] = (uint32_t)(run / 128);
            run = (run + (uint64_t)s->cells[c].count * rec_bytes + 127) / 128 * 128;
            if (run / 128 >= (1ull << 32)) return fail(SPH_ERR_RANGE, "buffer exceeds the 512 GiB offset range");
            ++n_sides;
        }
    }
    if (bytes_needed_out) *bytes_needed_out = run;
    if (!d_buf) return SPH_OK;             // size query: nothing is uploaded or launched
    if (buf_bytes < run) return fail(SPH_ERR_RANGE, "buffer of %llu bytes, %llu needed", (unsigned long long)buf_bytes, (unsigned long long)run);

    // occurrence lists: the blocks of each cell in ascending (task, side) order, cells ascending; one chunk table entry per
    // 32 particles of a touched cell.  Every table entry a launch reads is written here, so nothing is left from earlier calls.
    std::sort(h_key, h_key + n_sides);
    CellChunk* chunks = reinterpret_cast<CellChunk*>(h_tables + kChunksAt);
    double* frames = reinterpret_cast<double*>(h_tables + kFramesAt);
    uint32_t* off128 = reinterpret_cast<uint32_t*>(h_tables + kOffsetsAt);
    uint32_t n_chunks = 0;
    for (uint32_t o = 0; o < n_sides;) {
        const uint32_t c = (uint32_t)(h_key[o] >> 32);
        uint32_t o_end = o;
        while (o_end < n_sides && (uint32_t)(h_key[o_end] >> 32) == c) ++o_end;
        const sph_cell& ce = s->cells[c];
        const uint32_t need = (ce.count + 31) / 32;
        if (need > kMaxChunks - n_chunks)
            return fail(SPH_ERR_RANGE, "the cells of this call hold more than %u slices of 32 particles (SPH_PACK_STATIC_MAX_CHUNKS): split the bundle or use sph_batch_create + sph_pack",
                        kMaxChunks);
        for (uint32_t k = 0; k < ce.count; k += 32)
            chunks[n_chunks++] = CellChunk{(uint32_t)ce.first + k, std::min(32u, ce.count - k), k, o, o_end - o};
        for (; o < o_end; ++o) {
            const uint32_t side = (uint32_t)h_key[o], ts = h_side_task[side];
            const sph_task& tk = tasks[ts >> 1];
            std::memcpy(frames + 3 * (size_t)o, (ts & 1) ? tk.frame_j : tk.frame_i, 3 * sizeof(double));
            off128[o] = h_side_off128[side];
        }
    }
    if (n_chunks == 0) return SPH_OK;      // only empty cells: nothing to write

    unsigned char* d_scratch = nullptr;
    if (int32_t rc = scratch_address(&d_scratch)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // h_tables is ordinary (pageable) memory: each copy has left it by the time the call returns, so the lock may be dropped then
    SPH_CUDA_TRY(cudaMemcpyAsync(d_scratch + kChunksAt, chunks, (size_t)n_chunks * sizeof(CellChunk), cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(d_scratch + kFramesAt, frames, (size_t)n_sides * 3 * sizeof(double), cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(d_scratch + kOffsetsAt, off128, (size_t)n_sides * sizeof(uint32_t), cudaMemcpyHostToDevice, st));
    return launch_pack_tables(s->view(), prog, reinterpret_cast<const CellChunk*>(d_scratch + kChunksAt),
                              reinterpret_cast<const uint32_t*>(d_scratch + kOffsetsAt), reinterpret_cast<const double*>(d_scratch + kFramesAt),
                              (char*)d_buf, n_chunks, st);
    SPH_API_END
}
