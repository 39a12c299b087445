/* sph_b200.h -- C ABI of libsph_b200: the data-parallel hot path of the SPH GPU-offload pipeline of
 * arxiv/paper_2606_23891 ("Memory Layouts for GPU-Data Transfer Buffering in SPH"), B200 (sm_100a) only.
 *
 * Path (section 2.3, lines 76-82): per interaction loop, a bundle ("batch") of cell / cell-pair
 * tasks is PACKED (the attributes the loop reads are gathered out of the particle store into compact per-task
 * buffers), the loop runs on the buffers, and the results are UNPACKED (reduced) into the store.  The paper
 * packs and unpacks on the host CPU; here every step is a CUDA kernel.
 *
 * Conventions
 *  - every function returns an int32_t status (SPH_OK = 0); it never throws, aborts or prints;
 *    sph_last_error() returns the message of the calling thread's last failure.
 *  - "host" / "device" is stated for every pointer.  Handles (sph_store, sph_batch) are host objects that own
 *    device tables.  Transfer buffers are always DEVICE memory owned by the caller.
 *  - kernel-launching calls are asynchronous on the caller's stream (a cudaStream_t passed as void*; NULL = the
 *    legacy default stream).  Argument validation is synchronous and happens before any launch.
 *  - there is no CPU fallback: without a CUDA device every launching call returns SPH_ERR_CUDA.
 *
 * Data model (DESIGN.md gives the readings of the paper behind each choice)
 *  - particle: 18 fields / 26 scalar components, Table 1 of the paper completed by
 *    BASELINE.json:configs[0]; canonical exchange format = the 128-byte AoS record below.
 *  - store layout: a runtime descriptor (sph_layout): n_sub arrays of structs, each field lives in one
 *    substruct at one byte offset.  AoS = 1 substruct of 128 B; split-AoS = 6 substructs grouped
 *    by kernel read/write pattern (BASELINE.json:configs[1]).
 *  - cell: contiguous particle range [first, first+count).
 *  - task: one loop step on one cell (cj = -1) or on a cell pair; frame_i / frame_j are the
 *    points the two sides' coordinates are made relative to when packed (periodic shift).
 *  - attribute set: ordered list of field components; record = those components back to back, 4-byte units.
 *  - buffer of a batch: for each task in order: side-i block, then side-j block (pair tasks); a block holds
 *    `count` records in store order and starts at the next multiple of 128 bytes; pad bytes are unspecified.
 *    A batch created with tasks_per_segment = S lays its segments (chunks of S tasks) back to back, each
 *    segment starting at a multiple of 256 bytes and laid out exactly as a stand-alone batch of those tasks.
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    SPH_OK = 0,
    SPH_ERR_INVALID_ARG = 1,  /* NULL pointer, bad enum, inconsistent sizes */
    SPH_ERR_LAYOUT = 2,       /* layout descriptor or attribute set is malformed */
    SPH_ERR_RANGE = 3,        /* index / range / buffer size out of bounds */
    SPH_ERR_ALLOC = 4,        /* host or device allocation failed */
    SPH_ERR_CUDA = 5,         /* CUDA runtime error (no device, launch failure) */
    SPH_ERR_UNSUPPORTED = 6   /* valid request this build does not implement */
};

/* fields, in the member order of the canonical record */
enum {
    SPH_X = 0, SPH_V, SPH_A, SPH_MASS, SPH_H, SPH_U, SPH_DU_DT, SPH_RHO, SPH_RHO_DH, SPH_WCOUNT, SPH_WCOUNT_DH,
    SPH_DIV_V, SPH_ROT_V, SPH_P, SPH_CS, SPH_V_SIG, SPH_ID, SPH_TIME_BIN, SPH_NFIELDS
};

/* canonical 128-byte AoS record (natural C alignment):
 *   x f64[3] @0 | v f32[3] @24 | a f32[3] @36 | mass @48 | h @52 | u @56 | du_dt @60 | rho @64 | rho_dh @68 |
 *   wcount @72 | wcount_dh @76 | div_v @80 | rot_v f32[3] @84 | P @96 | c_s @100 | v_sig @104 | pad @108 |
 *   id i64 @112 | time_bin i8 @120 | pad @121..127 */
#define SPH_AOS_BYTES 128
#define SPH_MAX_SUB 8
#define SPH_MAX_ATTR 32

typedef struct {
    uint32_t n_sub;                 /* number of substruct arrays, 1..SPH_MAX_SUB */
    uint32_t stride[SPH_MAX_SUB];   /* bytes per particle in each substruct (multiple of 4) */
    struct { uint8_t sub; uint8_t pad; uint16_t off; } loc[SPH_NFIELDS];   /* home of each field */
} sph_layout;

typedef struct { uint8_t field, comp0, ncomp, pad; } sph_attr;   /* components [comp0, comp0+ncomp) of a field */

#define SPH_ATTR_X_REL_F32 1u   /* X is packed as (float)(x - frame): 4 bytes per component instead of 8 */

typedef struct {
    uint32_t n;                     /* entries used */
    uint32_t flags;                 /* SPH_ATTR_* */
    sph_attr ent[SPH_MAX_ATTR];     /* record = entries in this order, no padding.  Component sizes: X 8 bytes
                                       (4 with X_REL_F32), ID 8, TIME_BIN 4 (value in byte 0, bytes 1-3 zero),
                                       every other component 4 */
} sph_attrset;

/* the four canonical attribute sets of the density and force loops */
enum { SPH_SET_DENSITY_IN = 0,  /* [X(rel f32), H, MASS]                        20-byte record */
       SPH_SET_DENSITY_OUT = 1, /* [RHO, RHO_DH, WCOUNT, WCOUNT_DH]             16 */
       SPH_SET_FORCE_IN = 2,    /* [X(rel), H, MASS, RHO, RHO_DH, V, U, P, CS]  52 */
       SPH_SET_FORCE_OUT = 3,   /* [A, DU_DT, V_SIG]                            20 */
       /* the three-loop (Sphenix-like) cycle, PAPER.md:41 and Table 1 columns p-g / p-f (reading C34) */
       SPH_SET_GRADIENT_IN = 4, /* [X(rel), V, MASS, H, U, RHO]                 40 */
       SPH_SET_GRADIENT_OUT = 5,/* [DIV_V, ROT_V]                               16 */
       SPH_SET_FORCE3_IN = 6 }; /* FORCE_IN + [DIV_V, ROT_V, TIME_BIN]          72 */

typedef struct { uint64_t first; uint32_t count; uint32_t pad; double origin[3]; double width; } sph_cell;   /* 48 B */
typedef struct { int32_t ci, cj; double frame_i[3]; double frame_j[3]; } sph_task;                           /* 56 B */
typedef struct { float gamma, alpha, beta; } sph_params;   /* ideal-gas gamma; viscosity alpha, beta */

enum { SPH_MEM_DEVICE = 0, SPH_MEM_HOST_PINNED = 1 };
enum { SPH_UNPACK_REDUCE = 0,   /* per-field operator: += for the neighbour sums RHO, RHO_DH, WCOUNT, WCOUNT_DH, DIV_V, ROT_V, A,
                                   DU_DT; max for V_SIG; overwrite for every other field -- applied in ascending task
                                   order, side i before side j, in f32 (bit-reproducible) */
       SPH_UNPACK_ASSIGN = 1,   /* overwrite for every field, same order (last task wins) */
       SPH_UNPACK_REDUCE_ZERO = 2 }; /* SPH_UNPACK_REDUCE preceded by "zero the outputs" for the particles of the cells the call
                                   * touches: the sums start from 0 instead of the store's values (bit-identical to
                                   * sph_store_zero + SPH_UNPACK_REDUCE for those particles; others are left alone).  For the
                                   * first (or only) batch of a loop: saves a launch and the read of the fields. */

typedef struct sph_store sph_store;
typedef struct sph_batch sph_batch;

typedef struct {
    uint64_t n_tasks, n_self, n_pair;
    uint64_t n_sides;        /* task sides = blocks in a buffer */
    uint64_t n_instances;    /* sum of block particle counts */
    uint64_t n_candidates;   /* ordered candidate pairs the loops test: sum count_i*count_j (x2 for pair tasks) */
    uint64_t n_cells_touched;
    uint32_t n_segments;
    uint32_t max_count;      /* largest block */
    uint64_t n_items;              /* work items of an interaction loop: (<= 64 targets of a block) x (the block they gather from) */
    uint64_t max_item_candidates;  /* candidate pairs of the largest item: what one warp works through alone (load balance) */
} sph_batch_info;

/* ---- errors ---- */
/* Copies the calling thread's last error message (NUL-terminated, truncated to cap) into msg [host]. */
int32_t sph_last_error(char* msg, size_t cap);

/* ---- layouts and attribute sets (host only, BASELINE.json:configs[0..1]) ---- */
int32_t sph_layout_aos(sph_layout* out);     /* 1 substruct, the canonical 128-byte record */
int32_t sph_layout_split(sph_layout* out);   /* S0 {x,h,mass} 32 | S1 {rho,rho_dh,wcount,wcount_dh} 16 | S2 {v,u,P,c_s} 24 |
                                                S3 {a,du_dt,v_sig} 20 | S4 {id,time_bin} 16 | S5 {div_v,rot_v} 16 */
int32_t sph_layout_validate(const sph_layout* layout);   /* SPH_ERR_LAYOUT if fields overlap, misaligned or out of stride */
/* Any other struct split (random-order AoS, the kernel-driven sAoS variants, their splits by data
 * type): fields [host, n_fields <= SPH_NFIELDS field ids, every field exactly once] are laid out group by group,
 * group_sizes [host, n_groups <= SPH_MAX_SUB, sum = n_fields]; inside a substruct members follow one another in the given
 * order at their natural alignment (x, id: 8; time_bin: 1; else 4), the stride is rounded up to the largest member
 * alignment (at least 4) and to min_stride [host, n_groups strides or NULL] where given (e.g. 128 for a padded AoS record). */
int32_t sph_layout_from_groups(const uint8_t* fields, uint32_t n_fields, const uint32_t* group_sizes, uint32_t n_groups,
                               const uint32_t* min_stride, sph_layout* out);
int32_t sph_attrset_canonical(int32_t which, sph_attrset* out);
int32_t sph_attrset_record_bytes(const sph_attrset* set, uint32_t* bytes_out);   /* SPH_ERR_LAYOUT: a component listed twice */

/* ---- particle store ---- */
/* Bytes of substruct `sub` for n particles, including the 64 tail bytes the vectorised kernels may read. */
int32_t sph_store_sub_bytes(const sph_layout* layout, uint64_t n, uint32_t sub, uint64_t* bytes_out);
/* mem_kind: SPH_MEM_DEVICE (HBM) or SPH_MEM_HOST_PINNED (mapped pinned host memory the GPU reads/writes over
 * the host link).  ext_ptrs [host array of n_sub pointers] may name caller-owned memory of the right kind,
 * 256-byte aligned, sph_store_sub_bytes() long each (e.g. torch tensors); NULL: the store allocates and owns. */
int32_t sph_store_create(const sph_layout* layout, uint64_t n, int32_t mem_kind, void* const* ext_ptrs, sph_store** out);
int32_t sph_store_destroy(sph_store* store);
/* Canonical AoS in / out [host, n*128 bytes].  Synchronous.  export writes every byte of the canonical record
 * (pad bytes zero). */
int32_t sph_store_import_aos(sph_store* store, const void* host_aos, uint64_t n);
int32_t sph_store_export_aos(const sph_store* store, void* host_aos, uint64_t n);
/* Cell table [host]; ranges must lie inside the store and must not overlap.  Copied. */
int32_t sph_store_set_cells(sph_store* store, const sph_cell* cells, uint32_t n_cells);
int32_t sph_store_sub_ptr(const sph_store* store, uint32_t sub, void** ptr_out);
/* STAGING ("buffer contents are transferred to the GPU ... results are transferred back"): copy one
 * substruct array between the store and a host array in the store's own layout [host, n*stride bytes; pinned memory
 * makes the copy asynchronous on `stream`, pageable memory makes it synchronous].  With split-AoS only the
 * substructs a loop reads / writes have to cross the host link; with AoS the whole 128-byte records do. */
int32_t sph_store_upload_sub(sph_store* store, uint32_t sub, const void* host_src, uint64_t bytes, void* stream);
int32_t sph_store_download_sub(const sph_store* store, uint32_t sub, void* host_dst, uint64_t bytes, void* stream);
/* The same for the particles [first, first + count) of one substruct array: host_base [host] is the START of the host
 * array (n*stride bytes in the store's layout); bytes (first*stride .. (first+count)*stride) are copied.  Cells are
 * contiguous particle ranges, so the structs of a range of cells can cross the link while the kernels
 * work on the cells that crossed before (sph_pack_cells / sph_unpack_cells). */
int32_t sph_store_upload_range(sph_store* store, uint32_t sub, const void* host_base, uint64_t first, uint64_t count, void* stream);
int32_t sph_store_download_range(const sph_store* store, uint32_t sub, void* host_base, uint64_t first, uint64_t count, void* stream);

/* ---- cell grid / octree and task list (host, setup) ---- */
/* x3 [host, n*3 f64 in [0, box)].  perm_out [host, n]: perm_out[k] = input index of the k-th particle in cell
 * order (stable).  cells_out [host, cells_per_dim^3], row-major cell index (ix*n + iy)*n + iz. */
int32_t sph_cells_build_grid(const double* x3, uint64_t n, uint32_t cells_per_dim, double box, uint64_t* perm_out, sph_cell* cells_out);
/* Octree: a node is split while it holds more than max_per_leaf particles and every non-empty child stays at
 * least as wide as 2*hmax of its own particles.  Non-empty leaves in depth-first order (octant = 4bx+2by+bz).
 * *cells_out is allocated by the library (release with sph_free). */
int32_t sph_cells_build_octree(const double* x3, const float* h, uint64_t n, uint32_t max_per_leaf, double box,
                               uint64_t* perm_out, sph_cell** cells_out, uint32_t* n_cells_out);
/* One self task per cell (ascending), then pair tasks (ci < cj, sorted by (ci, cj)): (A, B) is a pair iff the
 * periodic minimum box-to-box gap is < max(2 hmax_A, 2 hmax_B).  frame_i = origin_ci, frame_j = origin_ci - s
 * (s = periodic image shift of cj).  SPH_ERR_RANGE if a second image is also within reach (box too small).
 * *tasks_out is allocated by the library (release with sph_free). */
int32_t sph_tasks_build(const sph_cell* cells, const float* hmax_per_cell, uint32_t n_cells, double box,
                        sph_task** tasks_out, uint64_t* n_self_out, uint64_t* n_pair_out);
int32_t sph_free(void* p);

/* ---- batches (bundles) ---- */
/* Builds the device tables of a batch of tasks [host array] against the store's cell table: block table, chunk tables,
 * per-cell occurrence lists for the cell-centric kernels.  tasks_per_segment = 0: one segment.  Immutable afterwards.
 * Synchronous.  The batch is tied to the cell table (not to the store object): it may be used with any store of the same
 * particle count whose cell table is the same (SPH_ERR_INVALID_ARG otherwise). */
int32_t sph_batch_create(const sph_store* store, const sph_task* tasks, uint64_t n_tasks, uint32_t tasks_per_segment, sph_batch** out);
int32_t sph_batch_destroy(sph_batch* batch);
int32_t sph_batch_get_info(const sph_batch* batch, sph_batch_info* info_out);
/* Bytes of the buffer that holds this batch for this attribute set.  A pure query: the batch is not changed as far as any
 * caller can observe (block offsets for a record size are derived from the immutable block table the first time any call
 * needs them, under a lock; sph_pack / sph_unpack accept any attribute set whether or not this was called). */
int32_t sph_batch_buffer_bytes(const sph_batch* batch, const sph_attrset* set, uint64_t* bytes_out);
/* Byte offset of every block for this attribute set: off_out [host, 2*n_tasks], off[2t] side i, off[2t+1] side j
 * (UINT64_MAX for self tasks).  seg_off_out [host, n_segments] may be NULL. */
int32_t sph_batch_block_offsets(const sph_batch* batch, const sph_attrset* set, uint64_t* off_out, uint64_t* seg_off_out);

/* ---- the hot path ---- */
/* Sets the listed f32 components of every particle to 0 ("zero the outputs of the loop about to run"). */
int32_t sph_store_zero(sph_store* store, const sph_attrset* set, void* stream);
/* PACK: for every block of the batch, gather the attribute set out of the store into
 * d_buf [device, buf_bytes >= sph_batch_buffer_bytes]; X with X_REL_F32 becomes (float)(x - frame_side). */
int32_t sph_pack(const sph_store* store, const sph_batch* batch, const sph_attrset* set, void* d_buf, uint64_t buf_bytes, void* stream);
/* DENSITY LOOP: d_in = DENSITY_IN buffer, d_out = DENSITY_OUT buffer of the same batch.  Per
 * instance i, over the other side (pair task) or the own cell including i (self task), with q = r/h_i, r < 2h_i:
 * rho += m_j W, rho_dh += m_j dW/dh, wcount += W, wcount_dh += dW/dh (cubic spline, support 2h). */
int32_t sph_density(const sph_batch* batch, const void* d_in, uint64_t in_bytes, void* d_out, uint64_t out_bytes, void* stream);
/* FORCE LOOP: d_in = FORCE_IN buffer, d_out = FORCE_OUT buffer: acceleration, du/dt and maximum
 * signal velocity with grad-h terms and Monaghan viscosity. */
int32_t sph_force(const sph_batch* batch, const void* d_in, uint64_t in_bytes, void* d_out, uint64_t out_bytes,
                  const sph_params* params, void* stream);
/* GRADIENT LOOP ("a third gradient loop between the density and the force loops"; reading C34):
 * d_in = GRADIENT_IN buffer, d_out = GRADIENT_OUT buffer.  Per instance i over j != i with r < 2 h_i:
 * g = (m_j / rho_j) dW/dr(r, h_i), e = (x_i - x_j) / r, dv = v_j - v_i:  div_v += g (dv . e), rot_v += g (e x dv). */
int32_t sph_gradient(const sph_batch* batch, const void* d_in, uint64_t in_bytes, void* d_out, uint64_t out_bytes, void* stream);
/* FORCE LOOP of the three-loop cycle: d_in = FORCE3_IN buffer, d_out = FORCE_OUT buffer; sph_force with the viscous term scaled
 * by (B_i + B_j) / 2, B = |div v| / (|div v| + |rot v| + 1e-4 c_s / h) (Balsara-type switch, reading C34). */
int32_t sph_force3(const sph_batch* batch, const void* d_in, uint64_t in_bytes, void* d_out, uint64_t out_bytes,
                   const sph_params* params, void* stream);
/* UNPACK: reduce / scatter the records of d_buf [device] into the store, mode = SPH_UNPACK_*.
 * X with X_REL_F32 cannot be unpacked (SPH_ERR_UNSUPPORTED). */
int32_t sph_unpack(sph_store* store, const sph_batch* batch, const sph_attrset* set, const void* d_buf, uint64_t buf_bytes,
                   int32_t mode, void* stream);
/* PACK / UNPACK restricted to the blocks of cells [cell_first, cell_first + cell_count) of the store's cell table
 * (every occurrence of those cells in the batch, at its place in d_buf; the other blocks are left alone).  Both kernels
 * are cell-centric -- a cell's particles are read (written) once and copied to (reduced from) all its blocks -- so
 * calls over disjoint cell ranges that cover the table are together exactly sph_pack / sph_unpack, and each call only
 * touches the store's particles of its own cells: the unit of the streamed host-resident path. */
int32_t sph_pack_cells(const sph_store* store, const sph_batch* batch, const sph_attrset* set, void* d_buf, uint64_t buf_bytes,
                       uint32_t cell_first, uint32_t cell_count, void* stream);
int32_t sph_unpack_cells(sph_store* store, const sph_batch* batch, const sph_attrset* set, const void* d_buf, uint64_t buf_bytes,
                         int32_t mode, uint32_t cell_first, uint32_t cell_count, void* stream);
/* ---- PACK without any allocation (for callers that must not call cudaMalloc) ----
 * sph_pack needs a batch, and sph_batch_create allocates device memory for the batch's tables.  Some hosts cannot do that
 * where they pack: a task-based SPH code (the paper's setting) takes its device memory once at start-up
 * and then runs many worker threads, each feeding its own stream -- a cudaMalloc / cudaFree inside a worker may wait for
 * the whole device and so stalls every other worker's stream, and on a GPU filled by the particle store it may just fail.
 * sph_pack_static is sph_pack for those callers: it takes the tasks themselves [host array, n_tasks entries] instead of a
 * batch, builds the tables for this one call in fixed host arrays, uploads them into a fixed scratch array inside the
 * library's device image (2.1 MiB per GPU that loads the library, held until the process exits) and launches the same pack
 * kernel.  It calls no cudaMalloc, cudaFree, cudaHostAlloc or other allocating routine, and uses no host heap.
 *  - store: any store; one created over caller memory (sph_store_create with ext_ptrs) never allocated device memory
 *    either.  set, d_buf [device, 128-byte aligned], stream: as sph_pack.  The buffer is laid out exactly as that of a
 *    one-segment batch of the same tasks (sph_batch_create with tasks_per_segment = 0), block bytes identical to sph_pack's.
 *  - bytes_needed_out [host, may be NULL]: receives the buffer size for these tasks and this set.  With d_buf = NULL the call
 *    is only that size query.
 *  - limits: n_tasks <= SPH_PACK_STATIC_MAX_TASKS, and the cells of the call together hold at most
 *    SPH_PACK_STATIC_MAX_CHUNKS slices of 32 particles (a cell of c particles counts ceil(c / 32), once however often it
 *    occurs).  Beyond either: SPH_ERR_RANGE before anything is uploaded or launched -- split the bundle.
 *  - the first call on each device looks up where the scratch array lives on that device (with that device current); make
 *    that first call during set-up, before any stream capture is begun.
 *  - ALL calls share the one scratch array.  A call overwrites every table entry its kernel reads, so nothing has to be
 *    cleared between calls, but two calls whose GPU work can overlap (different streams without an event between them, or
 *    two host threads on two streams) race: the later upload replaces tables the earlier kernel may still be reading.  Calls
 *    on one stream are safe, as are calls ordered by events.  On the host the calls of all threads take turns (a lock).
 *  - errors as sph_pack, plus the limits above; every call re-uploads its tables (36 bytes per block + 20 per slice), so
 *    where allocation is allowed sph_batch_create + sph_pack remains the faster path for a bundle that is packed repeatedly. */
#define SPH_PACK_STATIC_MAX_TASKS 16384u
#define SPH_PACK_STATIC_MAX_CHUNKS 65536u
int32_t sph_pack_static(const sph_store* store, const sph_task* tasks, uint32_t n_tasks, const sph_attrset* set, void* d_buf,
                        uint64_t buf_bytes, uint64_t* bytes_needed_out, void* stream);

/* ---- split pack loops ("loop fission", Fig. 4) ----
 * The paper splits the pack loop into several loops that each touch one substruct (by-struct), one quantity (by-element),
 * one data type (by-type) or one (substruct, type) pair.  GPU analogue: sph_pack_pass writes only the record words named in
 * word_mask (bit w = 4-byte word w of the record) for every block of the batch; the passes of a partition together write
 * exactly the bytes of sph_pack.  sph_pack_pass_masks gives the partition: split 0 by-struct, 1 by-element (one attribute
 * entry each), 2 by-type (f64 / f32 / i64 / i8), 3 by-struct-and-type; masks_out [host, >= 48], n_out [host] their number.
 * d_buf [device, 128-byte aligned, >= sph_batch_buffer_bytes]; asynchronous on stream; an empty mask is a no-op.  Errors, before
 * any launch: SPH_ERR_INVALID_ARG (NULL, misaligned, unknown split), SPH_ERR_RANGE (a mask bit beyond the record's words, buffer
 * too small), SPH_ERR_LAYOUT (bad attribute set). */
int32_t sph_pack_pass_masks(const sph_layout* layout, const sph_attrset* set, int32_t split, uint64_t* masks_out, uint32_t* n_out);
int32_t sph_pack_pass(const sph_store* store, const sph_batch* batch, const sph_attrset* set, uint64_t word_mask, void* d_buf,
                      uint64_t buf_bytes, void* stream);

/* ---- de-duplicated cell slots ("data replication") ----
 * A second input format for the loops: every cell the batch touches is packed ONCE into a slot (count records, slots in
 * ascending cell index, each starting at a multiple of 128 bytes) instead of once per task side (about 27 times on a
 * grid).  A slot record is the loop's input set with x as raw f64 plus time_bin as a last word: density [x f64[3], h,
 * mass, time_bin] 36 bytes, force [x f64[3], h, mass, rho, rho_dh, v, u, P, c_s, time_bin] 68 bytes (sph_slot_attrset).
 * The loop applies the frame of each task side itself, (float)(x - frame_side), exactly as sph_pack does, so
 * sph_density_slots / sph_force_slots write bit for bit the result buffers sph_density / sph_force write from per-task
 * buffers (which stay the parity format, reading C7); the result buffers and sph_unpack are unchanged.
 * loop: 0 density, 1 force.  d_slots, d_out [device, 128-byte aligned]; asynchronous on stream.  Errors as sph_pack / sph_density. */
int32_t sph_slot_attrset(int32_t loop, sph_attrset* out);
int32_t sph_batch_slot_bytes(const sph_batch* batch, int32_t loop, uint64_t* bytes_out);
int32_t sph_pack_slots(const sph_store* store, const sph_batch* batch, int32_t loop, void* d_slots, uint64_t slot_bytes, void* stream);
int32_t sph_density_slots(const sph_batch* batch, const void* d_slots, uint64_t slot_bytes, void* d_out, uint64_t out_bytes, void* stream);
int32_t sph_force_slots(const sph_batch* batch, const void* d_slots, uint64_t slot_bytes, void* d_out, uint64_t out_bytes,
                        const sph_params* params, void* stream);
/* GHOST: P = (gamma-1) rho u, c_s = sqrt(gamma (gamma-1) u) for every particle. */
int32_t sph_ghost(sph_store* store, const sph_params* params, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
