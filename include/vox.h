/*
 * vox.h -- C ABI of the B200 tetrahedral-mesh -> solid-binary-voxel library.
 *
 * What it computes (arxiv 2106.01326; citations are PAPER.md line numbers):
 *   "voxelizing the tetrahedral mesh according to whether the sampling point is
 *   within a tetrahedral or not": for every voxel-centre sample P
 *   of an nx*ny*nz grid and every tet whose bounding box covers P ("We iterate
 *   over every bounding box of the tetrahedral and apply the ... point-in-
 *   tetrahedral test") evaluate Theorem 1's four determinants
 *    and OR the result into a bit grid ("binary 3D grid",
 *   PAPER.md:110).
 *
 * Readings where the paper is silent:
 *   - the test is INCLUSIVE (closed tets);  tets with 6V == 0 contribute nothing;
 *   - sample = voxel centre  P = (hx*x + hx/2, hy*y + hy/2, hz*z + hz/2),
 *     h = extent / n per axis, on the integer lattice;
 *   - coordinates are int32 lattice points in [0, extent]; all predicates are
 *     evaluated in exact integer arithmetic (no floating point decides a bit).
 *
 * Grid layout (output of vox_run): for mesh m of the batch, voxel (x,y,z)
 *   word = ((m*nz + z)*ny + y)*(nx/32) + (x >> 5),  bit = x & 31  (LSB = lowest x),
 *   bit = 1 iff solid.  Every word of the grid is written by every vox_run.
 *
 * Memory ownership: ALL device memory is the caller's.  vox_tets borrows the
 * input pointers (no copy) until the last vox_run using them has completed on
 * its stream.  Workspace and output are caller-allocated.  The library
 * allocates only the host-side context.  vox_run only enqueues work on the
 * given stream: no allocation, no host synchronisation.
 *
 * Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  d_workspace must be
 * 16-byte aligned (VOX_EINVAL otherwise), d_tets 16-byte aligned, d_bits_out 4-byte aligned.
 * `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).
 *
 * Errors: every int-returning call returns VOX_OK (0) or a negative code;
 * nothing aborts or throws across the ABI.
 */
#ifndef VOX_H_
#define VOX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vox_ctx vox_ctx; /* opaque, host side */

enum {
    VOX_OK = 0,
    VOX_EINVAL = -1,     /* null pointer, n <= 0, nx % 32 != 0, extent % (2n) != 0, batch < 1, V/T < 0 */
    VOX_ERANGE = -2,     /* extent > 2^20 (the int64 bound 6*extent^3 < 2^63 would not hold), n > 32768,
                            more than 2^31-1 tiles */
    VOX_EWORKSPACE = -3, /* workspace too small (at enqueue, or reported by vox_status after a run) */
    VOX_ECUDA = -4,      /* CUDA runtime error; text via vox_last_error */
    VOX_ESTATE = -5,     /* call order: vox_run before vox_tets, ... */
    VOX_EDATA = -6       /* vox_validate: a vertex outside [0,extent] or a tet index outside [0,V) */
};

/* Grid dims in voxels (nx % 32 == 0), lattice extent per axis (extent % (2n) == 0
 * so that voxel centres are lattice points; extent <= 2^20), batch >= 1 meshes
 * sharing the grid shape. */
int vox_create(vox_ctx** out, int nx, int ny, int nz, int ex, int ey, int ez, int batch);
void vox_destroy(vox_ctx* ctx);

/* Optional: fix the binning tile (32 x ty x tz voxels; ty, tz powers of two in [4,32]).
 * Must precede vox_tets.  Without it vox_tets picks the tile from the grid and T (32^3
 * bricks for big grids, thinner tiles when that leaves too few or too heavy tiles).  The
 * result of vox_run does not depend on the tile; vox_tile_shape reports it. */
int vox_set_tile(vox_ctx* ctx, int ty, int tz);

/* Path variant, 0 = default.  Result-neutral by contract; only lattice input (vox_lattice) has a choice to make:
 *   0: the library picks: the binning passes K1-K3 (the faster device step on every measured workload of ordinary
 *      cells), the fused lattice path only when the mean cell is at least 64^3 voxels (giant cells);
 *   1: always the binning passes;
 *   2: the fused lattice path whenever the lattice is within its limits (see vox_lattice) -- the small-workspace
 *      variant: no range array, no pair list.
 * Any other value is refused with VOX_EINVAL (never silently ignored).  vox_path reports the path the next vox_run
 * takes: 0 = tet array through the binning passes, 1 = lattice input through the binning passes, 2 = lattice input
 * on the fused path (VOX_ESTATE before vox_tets / vox_lattice). */
int vox_set_variant(vox_ctx* ctx, int variant);
int vox_path(const vox_ctx* ctx);

/* Borrow the mesh.  d_verts int32[V][3] with coordinates in [0, extent];
 * d_tets int32[T][4], indices global into d_verts; d_tet_offsets int64[batch+1]
 * (device; mesh m owns tets [off[m], off[m+1]); off[0] = 0, off[batch] = T), or
 * NULL when batch == 1.  T == 0 is legal (all-zero grid).  Picks the binning tile unless
 * vox_set_tile fixed it (so workspace sizes and vox_tile_shape are valid after this call). */
int vox_tets(vox_ctx* ctx, const int32_t* d_verts, int64_t V, const int32_t* d_tets, int64_t T,
             const int64_t* d_tet_offsets);

/* Lattice input ("combining the background grid insertion method ... with the grid method for
 * voxelization sampling").  When the tet mesh IS a (jittered, carved) background lattice there is no
 * need for a tet array: d_verts int32[(cx+1)*(cy+1)*(cz+1)][3] holds the lattice vertices, vertex (i,j,k) at index
 * (i*(cy+1) + j)*(cz+1) + k; cell (i,j,k), index c = (i*cy + j)*cz + k, is split into the 6 Kuhn tets, tet q
 * walking from the cell's low corner along the axes of the q-th permutation of (x,y,z) in lexicographic order
 * (xyz, xzy, yxz, yzx, zxy, zyx); bit q of d_keep[c] says whether tet q is present.  Equivalent to vox_tets with
 * the 6*cx*cy*cz tets written out (absent ones dropped).  With batch > 1 every mesh has the same lattice dims:
 * mesh m's vertices and keep bytes are the m-th block of d_verts / d_keep.
 * vox_run on lattice input takes the binning passes over the implied tets by default (vox_set_variant above).  The
 * FUSED path (variant 2, or the default's own choice for giant cells): a pass over the vertices (K0) records, per axis and vertex plane
 * of the lattice, the coordinate range of the plane; each tile then finds the index box of the cells that can
 * reach it from those ranges and its own coordinates, enumerates their present tets and voxelizes them -- no
 * per-tet bbox search, no pair list, no K1/K2/K3 (the exact per-tet box inside the tile kernel keeps the result
 * the definition's).  Its workspace is the header, 8*(cx+cy+cz+3) bytes per mesh and a 16-byte copy of every vertex
 * (vox_workspace_bytes: on this path it is SMALLER than vox_workspace_fixed_bytes, which is what the optional vox_plan
 * needs -- the fused path has no pair list to size, so plan only if the pair count itself is wanted);
 * vox_status then reports culled = 0 (slivers and degenerate tets are skipped per tile, not counted per tet).
 * Lattices beyond 4096 cells per axis, 2^28 vertices or 65535 meshes take the binning passes whatever the variant
 * (vox_status then counts only present tets as culled).  vox_plan always runs the binning count. */
int vox_lattice(vox_ctx* ctx, const int32_t* d_verts, int cx, int cy, int cz, const uint8_t* d_keep);

/* batch * nz * ny * (nx/32) */
size_t vox_grid_words(const vox_ctx* ctx);

/* Workspace vox_run needs.  After vox_tets: the fixed part plus room for an
 * ESTIMATED number of (tet, brick) pairs (4*T + bricks).  After vox_plan: exact. */
size_t vox_workspace_bytes(const vox_ctx* ctx);
/* The part of the workspace that does not depend on the pair count (what vox_plan needs). */
size_t vox_workspace_fixed_bytes(const vox_ctx* ctx);

/* Optional exact sizing: runs the count + scan passes (K1, K2) on `cuda_stream`,
 * SYNCHRONISES it, and returns the number of (tet, brick) pairs.  Afterwards
 * vox_workspace_bytes is exact for this mesh.  Needs ws_bytes >= fixed bytes. */
int vox_plan(vox_ctx* ctx, void* cuda_stream, void* d_workspace, size_t ws_bytes, int64_t* pairs_out);

/* Enqueue the whole hot path (K1 count, K2 scan, K3 scatter, K4 brick voxelizer
 * with its large-tet path) on `cuda_stream`; writes every word of d_bits_out.
 * If the workspace cannot hold all pairs the excess tets are dropped and a device
 * flag is raised that vox_status reports. */
int vox_run(vox_ctx* ctx, void* cuda_stream, void* d_workspace, size_t ws_bytes, uint32_t* d_bits_out);

/* SYNCHRONISES the stream and reads the header the last vox_run left in the
 * workspace: returns VOX_EWORKSPACE if pairs were dropped; stats_out (may be
 * NULL) receives {pairs, culled tets (sliver or degenerate), large-path pairs,
 * non-empty bricks}. */
int vox_status(vox_ctx* ctx, void* cuda_stream, const void* d_workspace, int64_t stats_out[4]);

/* vox_run for callers that cannot allocate device memory.
 *
 * vox_run leaves the workspace to the caller, which normally means a cudaMalloc (or a framework tensor).  Some
 * callers of this library have no way to make one: a plug-in inside a host application whose own pool has
 * already claimed the whole GPU and which hands the plug-in nothing but its input and output buffers; a
 * service loop that must not stall its other streams (cudaMalloc and cudaFree synchronise the device); code
 * that runs while some other thread of the process is capturing a CUDA graph in the global capture mode,
 * where an allocation call is an error and ruins that capture.  For them the library carries its own
 * workspace: VOX_NOALLOC_SCRATCH_BYTES of device memory inside the library image, present on every GPU that
 * loads libvox.so from then until the process exits, whether or not this call is ever used.
 *
 * The call is vox_run with that built-in workspace: same kernels, same result, every word of d_bits_out
 * written.  The caller still passes the inputs (vox_tets / vox_lattice) and the output grid.  It calls no
 * cudaMalloc, cudaFree or any routine that allocates; it enqueues a memset and the kernels on `cuda_stream`.
 *
 *   Limit.   vox_workspace_bytes(ctx) must not exceed VOX_NOALLOC_SCRATCH_BYTES (4 MiB: roughly 24 bytes
 *            per tet plus 8 per tile, i.e. meshes up to ~150 000 tets on grids up to ~256^3; config 2 of
 *            BASELINE.json needs 1.9 MB).  Anything larger is refused with VOX_EWORKSPACE before any GPU
 *            work, and vox_last_error(ctx) says how many bytes were needed and how many there are.
 *   Set-up.  The first call on each device looks up that device's address of the built-in array
 *            (the device that is current at the call, which must be the one `cuda_stream` belongs to) and
 *            remembers it.  Make this first call before any stream capture begins.  Up to 64 devices.
 *   Sharing. There is ONE such array per device and every call on that device uses it, whatever the ctx,
 *            stream or thread.  Each call clears the counters it needs to start at zero itself, so stale
 *            contents from the previous call never matter; but two calls whose GPU work can overlap (different
 *            streams, no dependency between them) race on the array and both results are undefined.  Order
 *            them on one stream or with events.
 *   Status.  stats_out == NULL: enqueue only, as vox_run.  stats_out != NULL: the call then WAITS for the
 *            stream and fills stats_out like vox_status ({pairs, culled tets, large-path pairs, non-empty
 *            tiles}); it returns VOX_EWORKSPACE if the mesh produced more (tet, tile) pairs than the array
 *            had room for (tets were dropped: the grid is incomplete).  The estimate behind
 *            vox_workspace_bytes is not an upper bound, so pass stats_out at least once per kind of mesh. */
#define VOX_NOALLOC_SCRATCH_BYTES (4u << 20)
int vox_run_noalloc(vox_ctx* ctx, void* cuda_stream, uint32_t* d_bits_out, int64_t stats_out[4]);

/* Sparse (two-level) output.  "voxels are often calculated and stored in
 * octree data formats"; the binning tiles give a two-level store for free:
 * a table with one word per tile plus the row words of the MIXED tiles only.
 *
 *   tile t = ((m*nbz + bz)*nby + by)*nbx + bx  covers voxels x in [32bx, 32bx+32),
 *            y in [TY*by, TY*by+TY), z in [TZ*bz, TZ*bz+TZ) of mesh m  (vox_tile_shape gives
 *            {TY, TZ, nbx, nby, nbz}; nbx = nx/32, nby = ceil(ny/TY), nbz = ceil(nz/TZ));
 *   d_table[t] = 0            every voxel of the tile (inside the grid) is empty,
 *              = 0xFFFFFFFF   every voxel of the tile (inside the grid) is solid,
 *              = 1 + s        mixed: its row words are d_payload[s][z][y], z < TZ, y < TY
 *                             (same bit order as the dense grid; rows outside the grid are 0),
 *              = 0xFFFFFFFE   mixed but dropped: payload capacity exceeded (VOX_EWORKSPACE
 *                             from vox_sparse_status / vox_pipe_wait).
 * The slots s of the mixed tiles are a permutation of 0..mixed-1 in no particular order; the
 * decoded grid is unique and equals vox_run's.  d_table has NB = batch*nbz*nby*nbx words,
 * d_payload payload_capacity_tiles * TY*TZ words; d_payload may be the device view of pinned
 * host memory.  vox_sparse_status SYNCHRONISES and returns {mixed tiles, full tiles} of the
 * last vox_run_sparse on this workspace. */
int vox_tile_shape(const vox_ctx* ctx, int out[5]);
int vox_run_sparse(vox_ctx* ctx, void* cuda_stream, void* d_workspace, size_t ws_bytes, uint32_t* d_table,
                   uint32_t* d_payload, int64_t payload_capacity_tiles);
int vox_sparse_status(vox_ctx* ctx, void* cuda_stream, const void* d_workspace, int64_t out[2]);

/* Occupancy from sub-samples.  The paper's comparison voxelizes "each model ... into 5
 * million samples, with a resolution of 256^3": more than one sample per voxel.  Reading taken
 * (DESIGN.md): k x k x k regularly spaced sub-samples per voxel = the voxel centres of a grid k times finer per
 * axis, so the mesh is voxelized with vox_run on (k*nx, k*ny, k*nz) and this call folds that bit grid:
 *   d_counts_out[((m*nz + z)*ny + y)*nx + x] = number of solid sub-samples of voxel (x,y,z), 0..k^3 (uint8).
 * nx, ny, nz are the COARSE dims; k is 2 or 4; (k*nx) % 32 == 0; d_bits_fine has the vox_run layout of the fine
 * grid.  Enqueue only (no sync, no allocation). */
int vox_occupancy(void* cuda_stream, const uint32_t* d_bits_fine, int nx, int ny, int nz, int batch, int k,
                  uint8_t* d_counts_out);

/* Debug: device pass + sync; VOX_EDATA if a vertex lies outside [0,extent] or a
 * tet index outside [0,V) or the offsets are not monotone.  d_workspace needs
 * only the fixed part. */
int vox_validate(vox_ctx* ctx, void* cuda_stream, void* d_workspace, size_t ws_bytes);

/* End-to-end convenience for HOST buffers, one mesh, fully serialised (vox_pipe_* below overlaps the copies):
 * copies h_verts / h_tets / h_tet_offsets into the caller's device arena, runs
 * vox_tets + vox_run on `cuda_stream`, copies the grid to h_bits_out and
 * synchronises.  Host buffers should be pinned.  Arena layout is private;
 * vox_host_arena_bytes(ctx, V, T) says how large it must be (it includes an
 * estimated-pairs workspace; pass a larger arena for pathological meshes).
 * Returns VOX_EWORKSPACE if pairs were dropped. */
size_t vox_host_arena_bytes(const vox_ctx* ctx, int64_t V, int64_t T);
int vox_run_host(vox_ctx* ctx, void* cuda_stream, const int32_t* h_verts, int64_t V,
                 const int32_t* h_tets, int64_t T, const int64_t* h_tet_offsets,
                 void* d_arena, size_t arena_bytes, uint32_t* h_bits_out);

/* Transfer-overlapped pipeline for a STREAM of meshes in host memory.
 * The paper's own tables say the host<->device copies, not the kernel, dominate
 * ("the overhead of copying data to GPU memory"; Table 2),
 * so consecutive meshes are overlapped: while mesh k is voxelized, mesh k+1 is copied in
 * and grid k-1 is copied out, on three internal non-blocking streams, `depth` meshes in
 * flight.  Every mesh runs exactly the vox_tets + vox_run path above.
 *
 *   vox_pipe_create   grid/extent/batch as vox_create; depth in [1,8]; max_V/max_T bound
 *                     the meshes that will be submitted.  Creates streams, events and a
 *                     small pinned status block per slot (host-side allocations: call it
 *                     outside any timed region).
 *   vox_pipe_arena_bytes  device bytes the caller must provide (depth x [verts, tets,
 *                     offsets, grid, estimated-pairs workspace]).
 *   vox_pipe_reserve_pairs  optional, before vox_pipe_bind: size every slot's pair list for
 *                     max_pairs (tet, tile) pairs instead of the estimate 4*max_T + tiles (meshes
 *                     of large tets on small tiles exceed it; vox_plan gives the exact number).
 *   vox_pipe_bind     hand over the caller's device arena (borrowed until destroy).
 *   vox_pipe_submit   enqueue one mesh: H2D of h_verts int32[V][3], h_tets int32[T][4],
 *                     h_tet_offsets int64[batch+1] (NULL if batch == 1), the hot path,
 *                     D2H of the grid into h_bits_out (uint32[vox_grid_words]).  Host
 *                     buffers must be pinned and stay untouched until the ticket is
 *                     waited on.  Blocks only when all `depth` slots are in flight (then
 *                     it waits for the oldest).  *ticket_out = 0,1,2,... in submit order.
 *   vox_pipe_wait     block until that mesh's grid is in h_bits_out; VOX_EWORKSPACE if
 *                     pairs were dropped (arena workspace too small for this mesh);
 *                     stats_out (6 values, see below; may be NULL).  Tickets may be waited once,
 *                     in any order, but no later than `depth` submits after their own.
 *   vox_pipe_submit_sparse  as vox_pipe_submit with the sparse output of vox_run_sparse:
 *                     h_table uint32[NB] is copied out after the run; the mixed tiles are stored
 *                     by the kernel itself straight into h_payload (pinned, device-mapped host
 *                     memory, payload_capacity_tiles * TY*TZ words), so there is no separate
 *                     grid copy at all.
 *   vox_pipe_set_variant / vox_pipe_set_tile / vox_pipe_tile_shape  as the vox_ctx calls.
 * stats_out of vox_pipe_wait: {pairs, culled tets, large-path pairs, non-empty tiles,
 * mixed tiles, full tiles} (the last two only after a sparse submit).
 */
typedef struct vox_pipe vox_pipe;
int vox_pipe_create(vox_pipe** out, int nx, int ny, int nz, int ex, int ey, int ez, int batch, int depth,
                    int64_t max_V, int64_t max_T);
void vox_pipe_destroy(vox_pipe* pipe);
int vox_pipe_set_variant(vox_pipe* pipe, int variant);
int vox_pipe_set_tile(vox_pipe* pipe, int ty, int tz);
int vox_pipe_reserve_pairs(vox_pipe* pipe, int64_t max_pairs);
size_t vox_pipe_arena_bytes(const vox_pipe* pipe);
int vox_pipe_bind(vox_pipe* pipe, void* d_arena, size_t arena_bytes);
int vox_pipe_submit(vox_pipe* pipe, const int32_t* h_verts, int64_t V, const int32_t* h_tets, int64_t T,
                    const int64_t* h_tet_offsets, uint32_t* h_bits_out, int64_t* ticket_out);
int vox_pipe_submit_sparse(vox_pipe* pipe, const int32_t* h_verts, int64_t V, const int32_t* h_tets, int64_t T,
                           const int64_t* h_tet_offsets, uint32_t* h_table, uint32_t* h_payload,
                           int64_t payload_capacity_tiles, int64_t* ticket_out);
/* Lattice input through the pipe (vox_lattice): h_verts int32[(cx+1)(cy+1)(cz+1)][3] and h_keep uint8[cx*cy*cz],
 * pinned.  payload_capacity_tiles < 0: dense (h_out = the grid); otherwise sparse (h_out = tile table, h_payload as
 * in vox_pipe_submit_sparse).  The pipe must have been created with max_T >= batch*6*cx*cy*cz and
 * max_V >= batch*(cx+1)(cy+1)(cz+1). */
int vox_pipe_submit_lattice(vox_pipe* pipe, const int32_t* h_verts, int cx, int cy, int cz, const uint8_t* h_keep,
                            uint32_t* h_out, uint32_t* h_payload, int64_t payload_capacity_tiles, int64_t* ticket_out);
int vox_pipe_wait(vox_pipe* pipe, int64_t ticket, int64_t stats_out[6]);
int vox_pipe_tile_shape(const vox_pipe* pipe, int out[5]);
const char* vox_pipe_last_error(const vox_pipe* pipe);

/* Benchmark instrumentation (off by default).  vox_timing_enable(ctx, slots > 0)
 * creates a ring of CUDA events (a host-side allocation: call it outside any timed
 * region); every later vox_run then records an event on its stream before K1's
 * memset and after each of K1, K2, K3, K4 (no synchronisation).  Runs are numbered
 * 0,1,2,... from the enable call.  vox_timing_read(ctx, run, ms) returns the
 * durations {K1 incl. memset, K2, K3, K4, whole run} in milliseconds of a run that
 * has COMPLETED (the caller synchronises) and is still in the ring, else VOX_ESTATE.
 * A vox_run enqueued on a stream that is being captured into a CUDA graph records no events
 * and takes no run number.  slots == 0 disables and frees. */
int vox_timing_enable(vox_ctx* ctx, int slots);
int vox_timing_read(vox_ctx* ctx, int run, float ms_out[5]);

/* Roofline probe (not on the hot path): enqueue a dependent-free integer kernel
 * on `cuda_stream`.  kind 0 = IADD3/LOP3 stream (alu pipe), 1 = IMAD stream
 * (fma pipe), 2 = mixed.  *ops_out = thread-level INT32 ops it executes. */
int vox_probe_int32(void* cuda_stream, int kind, int blocks, int iters, uint32_t* d_sink,
                    double* ops_out);

/* Number of CUDA kernels this library has launched in this process so far (all contexts and pipes; memsets and
 * copies are not kernels).  bench.py reports the difference across its timed region as `gpu_launches`. */
uint64_t vox_kernel_launches(void);

/* Checked build (libvox_checked.so, compiled with -DVOX_CHECKS by paper_2106_01326_b200.build.build_checked): every
 * index the kernels form (tile ids, list entries, vertex ids, record slots, image-row addresses, queue slots, grid
 * words) is tested before use and the code of the first violated check is kept on the device.  SYNCHRONISES the
 * device, returns 1 and stores that code (0 = none) in *code_out, then clears it; the normal library compiles no
 * check and returns 0.  Test instrumentation: compute-sanitizer is closed on this pool (profiles/r02_sanitizers.md). */
int vox_debug_check_status(uint32_t* code_out);

/* Checked build only (the normal library compiles no test kernel and returns 0): runs the integer helpers the row
 * walk of K4 is built on over caller-supplied operand arrays, one element per thread, so that a test can compare them
 * with exact integer division operand by operand instead of through whole meshes (a compiler mis-fold corrupted
 * exactly this code twice).  d_a, d_b int64[n], d_out int32[n], all on the device; enqueue only.
 *   op 0: span_bound(r = a, mx = -b, inv = recip_up(b))      the per-row bound with the fast set-up's reciprocal
 *   op 1: span_bound(r = a, mx = -b, inv = 0xFFFFFFFF/b + 1)  the same with the general set-up's exact reciprocal
 *         contract (4 <= b < 2^31, |a|(1 + 2^-18) + b < 2^31): a >= 0 and a/b < 2^18 -> floor(a/b); a/b >= 2^18 -> some
 *         value >= 2^18 - 1; a < 0 -> some value <= -1
 *   op 2: (a * div_magic(b)) >> 16 = a / b for 0 <= a < 1024, 1 <= b <= 32   (row index -> slice of the local box)
 *   op 3: span64_bound(q0 = a, a = b) = max{x in [0,31] : q0 - b*x >= 0} or -1   (int64 large path)
 *   op 4: recip_up(b): in [2^32/b, (2^32/b)(1 + 2^-19) + 1), never below 2^32/b
 * Returns 1 when the kernel was enqueued, 0 in the normal build, a negative code on bad arguments. */
int vox_debug_selftest(void* cuda_stream, int op, const int64_t* d_a, const int64_t* d_b, int64_t n, int32_t* d_out);

const char* vox_strerror(int code);
const char* vox_last_error(const vox_ctx* ctx); /* CUDA error text of the last VOX_ECUDA */

#ifdef __cplusplus
}
#endif
#endif /* VOX_H_ */
