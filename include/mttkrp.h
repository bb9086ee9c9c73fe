/*
 * mttkrp.h - C-ABI of libmttkrp_b200: all-mode sparse MTTKRP with dynamic tensor remapping
 * on one NVIDIA B200 (sm_100a).
 *
 * The operation (arxiv 2405.08470; citations are PAPER.md line numbers):
 *   Y_d[i_d, r] = sum over nonzeros k of val_k * prod_{m != d} A_m[i_m(k), r]
 *     - Eq. 1 and the elementwise form of Sec. 2.1.5;
 *     - Alg. 2 "Elementwise Computation for mode d";
 *     - Alg. 3 "Dynamic Tensor Remapping": before mode d the nonzeros are
 *       re-ordered into the mode-d layout, in which all nonzeros of one output row are adjacent
 *       (Observation 2) and every element has a unique position
 *       (Observation 1);
 *     - Alg. 5: for d = 0..N-1 { compute mode d; barrier; swap(T_in, T_out) }.
 *
 * Conventions (all entry points):
 *   - Every call returns a status; nothing throws, aborts or prints.  mttkrp_last_error() gives a
 *     thread-local message for the last non-OK status.
 *   - "device" pointers are CUDA device memory of the current device, "host" pointers are ordinary
 *     host memory.  Device pointers must be 16-byte aligned.
 *   - The library never allocates device memory: the caller passes one workspace (size from
 *     mttkrp_workspace_bytes) which the handle borrows until mttkrp_destroy.
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = default stream).  mttkrp_mode and
 *     mttkrp_sweep are asynchronous on that stream; mttkrp_create synchronises the stream because
 *     it reads back counts and the index-error flag.
 *   - Indices are 0-based.  Duplicate coordinates are legal and add.  nnz == 0 is legal.
 *   - There is no CPU fallback: without a CUDA device every compute call returns MTTKRP_ECUDA.
 *   - A handle is not thread-safe; distinct handles are independent.
 *   - Calls on one handle execute in call order even when they are given different streams: the handle
 *     remembers the stream of its last call and makes a call on another stream wait (cudaStreamWaitEvent) for
 *     the work launched before it.  The caller still orders its own use of `out` and of the factor buffers.
 *   - Process environment variables (test and experiment knobs; unset = the library decides).  They are read in one
 *     place, by mttkrp_workspace_bytes and mttkrp_create, and checked BEFORE anything is launched: a malformed value
 *     is MTTKRP_EINVAL with the variable named in mttkrp_last_error(), never a silent default.  0|1 switches accept
 *     exactly "0" or "1"; numbers are decimal integers with nothing after them.  The handle keeps the values it was
 *     created with; they must not change between the size query and create.
 *       MTTKRP_KEY_ORDER = revcyclic|desc|asc|cyclic      sort-key order of the layouts
 *       MTTKRP_PACK = 0|1                                 0: 4*(nmodes+1)-byte records even where 16-byte packing fits
 *       MTTKRP_REMAP_BLOCKED = 0|1                        pin the blocked remap walk off / on for every transition
 *       MTTKRP_REMAP_BLOCK_LOG2 = integer                 log2 records per source block, clamped to [10,26]
 *       MTTKRP_REMAP_TWOPASS = 0|1                        pin the two-pass remap walk off / on.  Unpinned, create
 *                                                         TIMES both walks on the real tensor (median of 3 runs each)
 *                                                         and keeps the faster per transition, so on a busy GPU the
 *                                                         choice in info.remap_blocked can differ between runs (the
 *                                                         results never do); pin it for reproducible timings
 *       MTTKRP_TWOPASS_WINDOW_LOG2 = integer              log2 records per destination window, clamped to [8,26]
 *       MTTKRP_FORCE_DEEP = 0|1                           pin the MTTKRP kernel variant (nmodes <= 3)
 *       MTTKRP_PREFETCH_ROWS = integer >= 0               rows per factor matrix that are NOT prefetched into L2
 *                                                         (default 65536; 0 = no prefetch)
 *       MTTKRP_FUSE = 0|1                                 1: the remap runs inside the MTTKRP kernel.  Needs 16-byte
 *                                                         records (nmodes == 3, or packed nmodes >= 4) and the default
 *                                                         shard policy; asked for elsewhere it is MTTKRP_EUNSUPPORTED
 *       MTTKRP_SHARD_POLICY = equal|alg1                  alg1: the paper's Alg. 1 partitioner
 *       MTTKRP_KAPPA = integer in [1,65536]               partitions of the alg1 policy (default one per SM)
 */
#ifndef MTTKRP_B200_H
#define MTTKRP_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MTTKRP_MAX_MODES 8

typedef struct mttkrp_handle_s* mttkrp_handle_t; /* opaque host object */

typedef enum {
    MTTKRP_OK = 0,
    MTTKRP_EINVAL = 1,       /* bad argument (null pointer, size, mode, rank, alignment) */
    MTTKRP_EINDEX = 2,       /* an index is outside [0, dims[m]) (detected on the device in create) */
    MTTKRP_EUNSUPPORTED = 3, /* nmodes outside [2,8], R not in {8,16,32,64}, nnz >= 2^31, a dimension >= 2^28 */
    MTTKRP_EWORKSPACE = 4,   /* workspace too small or misaligned */
    MTTKRP_ECUDA = 5         /* a CUDA runtime call or kernel launch failed */
} mttkrp_status_t;

/* What a handle holds; filled by mttkrp_get_info (host struct). */
typedef struct {
    int32_t nmodes;
    int32_t cur_layout;                  /* mode whose order the resident tensor copy is in (0 after create) */
    int64_t nnz;
    int64_t dims[MTTKRP_MAX_MODES];
    int32_t record_bytes;                /* bytes per nonzero in the device format: 16 for nmodes == 3 and for the
                                            bit-packed records of nmodes >= 4, else 4*(nmodes+1) */
    int32_t shard_nnz;                   /* nonzeros per thread-block shard */
    int64_t num_shards;                  /* ceil(nnz / shard_nnz); same for every mode */
    int64_t num_split_rows[MTTKRP_MAX_MODES];  /* output rows whose nonzeros span more than one shard */
    int64_t num_empty_rows[MTTKRP_MAX_MODES];  /* output rows with no nonzero (stored as zeros) */
    int64_t bytes_held;                  /* device bytes the handle keeps after create (both tensor copies, maps, tables,
                                            staging for the *_host entry points): the handle uses workspace[0, bytes_held)
                                            and never touches the bytes from bytes_held on once mttkrp_create has returned,
                                            so the caller may reuse them.  It is below mttkrp_workspace_bytes by the
                                            create-time scratch and by the walk maps (8 bytes per nonzero) of every
                                            remap transition whose measured walk turned out to be the plain one */
    int64_t bytes_paper_format;          /* FLYCOO bytes by the paper's formula, PAPER.md:187:
                                            nnz * (N*ceil(log2 nnz) + sum ceil(log2 I_h) + 32) / 8 */
    int64_t remaps_done;                 /* remap passes executed since create */
    int32_t key_order[MTTKRP_MAX_MODES][MTTKRP_MAX_MODES];
                                         /* key_order[d] = sort-key order of the mode-d layout:
                                            key_order[d][0] == d, then the other modes (major to minor) */
    int32_t remap_blocked[MTTKRP_MAX_MODES];
                                         /* walk of the remap d -> (d+1)%N: 0 plain (destination order), 1 blocked (destination
                                            visited in source-block order: L2-resident gather window), 2 two passes (records
                                            first grouped by 32 MB destination window, then gathered inside the window) */
    double remap_avg_run[MTTKRP_MAX_MODES];
                                         /* average length of the ascending destination runs of that walk */
    int32_t shard_policy;                /* 0: equal-nnz shards, rows may span blocks (default); 1: the paper's Alg. 1
                                            (PAPER.md:163-181): whole rows dealt to kappa partitions, one block each */
    int32_t kappa;                       /* partitions of the Alg. 1 policy (0 under the default policy) */
    int64_t max_partition_nnz[MTTKRP_MAX_MODES];   /* Alg. 1 policy: largest / smallest partition per mode, in nonzeros */
    int64_t min_partition_nnz[MTTKRP_MAX_MODES];
    double remap_plain_ms[MTTKRP_MAX_MODES];       /* create-time measurement (median of 3 runs) of the plain and of the two-pass */
    double remap_twopass_ms[MTTKRP_MAX_MODES];     /* walk of that transition on this tensor (0: two passes were not a candidate) */
    int32_t fused_remap;                 /* 1: MTTKRP_FUSE=1 is in effect - the MTTKRP kernel of mode d also scatters the
                                            records into the layout of mode (d+1)%N (Alg. 4 lines 15-19) */
    int32_t reserved_;
    int64_t cold_rows[MTTKRP_MAX_MODES]; /* cold-row marks (nmodes <= 3): rows of mode m that are NOT among the
                                            MTTKRP_PREFETCH_ROWS most frequent ones (0: the factor has no cold row); the
                                            MTTKRP kernel requests such rows into L2 ahead of their gathers */
    int64_t cold_degree[MTTKRP_MAX_MODES];/* ... a row of mode m is cold when its index occurs fewer than this many times */
} mttkrp_info_t;

/*
 * Device workspace the handle needs for a tensor of this shape (pure host arithmetic).
 * max_rank: largest R that will be used with the *_host entry points (staging for factors and
 * output is then included); pass 0 if only device-pointer entry points are used.
 */
mttkrp_status_t mttkrp_workspace_bytes(int nmodes, const int64_t* dims /*host*/, int64_t nnz,
                                       int max_rank, size_t* bytes /*host, out*/);

/*
 * Build the device format from COO (Sec. 3.2/3.5 PAPER.md:147-149,183-189 as behaviour; the
 * layout itself is this library's): for every mode d a stable sort of the nonzeros by the key
 * tuple key_order[d] (output index first), the position maps between consecutive layouts (the
 * paper's remap ids), the empty-row and split-row tables, and the tensor copy in
 * mode-0 order (Alg. 5 input PAPER.md:308).
 *
 *   idx   device int32 [nmodes][nnz] (SoA, idx[m*nnz + k]), vals device fp32 [nnz], dims host.
 *   The COO arrays are only read, and are no longer needed once the call returns.
 *   workspace: device, >= mttkrp_workspace_bytes(...), borrowed until destroy.
 * Errors: EINVAL / EUNSUPPORTED / EWORKSPACE before any launch; EINDEX if an index is out of
 * range; ECUDA.  On error *out is NULL and the workspace contents are undefined.
 */
mttkrp_status_t mttkrp_create(mttkrp_handle_t* out, int nmodes, const int64_t* dims, int64_t nnz,
                              const int32_t* idx, const float* vals, int max_rank,
                              void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Y_d = MTTKRP along mode d (Alg. 2 + Alg. 3 + one iteration of Alg. 5's loop).
 *   factors: host array of nmodes device pointers; A_m is fp32 [dims[m]][R] row-major (ld = R).
 *            factors[d] is not read and may be NULL.
 *   out:     device fp32 [dims[d]][R] row-major; fully overwritten (rows without nonzeros get 0).
 *            Must not alias a factor that is read.
 *   Any d in any order.  If the resident layout is not d the tensor is first remapped: one gather pass
 *   (the cyclic order of Alg. 5, d == cur+1, uses the stored walk; any other d first composes the stored
 *   position maps into one direct map cur -> d, cached for the next identical jump).
 */
mttkrp_status_t mttkrp_mode(mttkrp_handle_t h, int d, const float* const* factors, int R,
                            float* out, void* cuda_stream);

/* All modes d = 0..nmodes-1 in order (Alg. 5).  outs: host array of nmodes
 * device pointers, outs[d] as `out` above.  Factors are not updated between modes. */
mttkrp_status_t mttkrp_sweep(mttkrp_handle_t h, const float* const* factors, int R,
                             float* const* outs, void* cuda_stream);

/* Only the remap pass into layout d (Alg. 3), no computation; used to time the two separately
 * and by tests. */
mttkrp_status_t mttkrp_remap_to(mttkrp_handle_t h, int d, void* cuda_stream);

/*
 * Same as mttkrp_sweep with HOST buffers: factors[m] host fp32 [dims[m]][R] (pinned memory makes
 * the copies asynchronous), outs[d] host fp32 [dims[d]][R].  Copies every factor to the
 * workspace staging area, runs all modes, copies every Y_d back, and synchronises before
 * returning.  The copies run on two internal streams so that they overlap the kernels (the
 * kernels run on cuda_stream).  Needs max_rank >= R at create.
 */
mttkrp_status_t mttkrp_sweep_host(mttkrp_handle_t h, const float* const* factors, int R,
                                  float* const* outs, void* cuda_stream);

/* Frees the host object.  Blocks until the work this handle launched has finished (the workspace is the
 * caller's again on return); touches no device memory itself. */
mttkrp_status_t mttkrp_destroy(mttkrp_handle_t h);

/* Thread-local message of the last failing call ("" if none). */
const char* mttkrp_last_error(void);

/* Introspection for tests and reports. */
mttkrp_status_t mttkrp_get_info(mttkrp_handle_t h, mttkrp_info_t* info /*host, out*/);

/* perm_dev[k] (device uint32 [nnz]) = original COO position of the nonzero at position k of the
 * mode-d layout, i.e. the stable sort permutation for key_order[d] (Observation 1).
 * scratch_dev: device uint32 [nnz], clobbered.  Asynchronous on cuda_stream. */
mttkrp_status_t mttkrp_get_perm(mttkrp_handle_t h, int d, uint32_t* perm_dev, uint32_t* scratch_dev,
                                void* cuda_stream);

/*
 * mttkrp_get_perm without the caller's scratch buffer, for callers that cannot allocate device memory when they call.
 *
 * Who that is: code hosted by an application whose own memory pool has already taken the GPU's memory (a raw
 * cudaMalloc there fails for lack of memory the pool is sitting on, and if it succeeds the pool's accounting no
 * longer matches the device), and code on a multi-stream pipeline that cannot afford the device-wide stall that
 * cudaMalloc and cudaFree bring.  mttkrp_get_perm asks such a caller for a second nnz-word buffer it has no way to
 * produce.  Here that buffer is a fixed array inside the library image instead; the call itself uses no cudaMalloc,
 * no cudaFree and no library routine that allocates.
 *
 *   perm_dev: device uint32 [nnz], the output, exactly as mttkrp_get_perm writes it (bit for bit).
 *   Limit:    nnz <= MTTKRP_NOALLOC_MAX_NNZ (4,194,304 nonzeros; the array is 16 MiB).  A larger handle gets
 *             MTTKRP_EUNSUPPORTED and nothing is launched; use mttkrp_get_perm for it.
 *   Cost:     every GPU on which this library is loaded holds those 16 MiB until the process ends, used or not.
 *   Set-up:   the first call on a device looks up the array's device address (once per device; the handle's device
 *             must be current, else MTTKRP_EINVAL).  Make that first call before any stream capture begins.
 *   Sharing:  all calls on one device use the same array.  Calls on the same stream are ordered and safe; two calls
 *             that can overlap on the GPU (different streams without a dependency, different handles or host
 *             threads) race on it and may return wrong permutations - serialise them yourself.  The array keeps
 *             what the last call left in it; that is harmless, because every word a call reads it has written
 *             first, so nothing needs to start at zero.
 * Asynchronous on cuda_stream.  Errors: EINVAL (NULL handle / perm_dev, d out of range, wrong current device),
 * EUNSUPPORTED (nnz over the limit, device ordinal >= 64), ECUDA.
 */
#define MTTKRP_NOALLOC_MAX_NNZ (1 << 22)
mttkrp_status_t mttkrp_get_perm_noalloc(mttkrp_handle_t h, int d, uint32_t* perm_dev, void* cuda_stream);

/* Copy the resident tensor copy out as SoA COO in its current layout order (device int32
 * [nmodes][nnz] in ORIGINAL mode numbering, device fp32 [nnz]).  Test hook for the remap. */
mttkrp_status_t mttkrp_export_coo(mttkrp_handle_t h, int32_t* idx_dev, float* vals_dev, void* cuda_stream);

/*
 * Optional per-kernel-class timing for reports (bench.py's roofline figure).  Between begin and end
 * the library records a CUDA event pair around every kernel it launches for this handle, on the
 * stream the kernel is launched on.  end synchronises cuda_stream, sums the elapsed times per class
 * and stops recording.  Off by default; adds two event records per launch while on.
 */
typedef struct {
    double remap_ms, zero_ms, mttkrp_ms, fixup_ms;                 /* summed device time per kernel class */
    int64_t remap_launches, zero_launches, mttkrp_launches, fixup_launches;
} mttkrp_timing_t;
mttkrp_status_t mttkrp_timing_begin(mttkrp_handle_t h);
mttkrp_status_t mttkrp_timing_end(mttkrp_handle_t h, mttkrp_timing_t* out /*host*/, void* cuda_stream);

/*
 * The paper's tensor partitioning scheme for one mode (Alg. 1), as an analysis tool: the
 * output rows of mode d ("vertices", with degree = number of nonzeros in the row) are ordered by descending
 * degree (ties: lower index first) and dealt one by one to the currently least-loaded of kappa partitions
 * (ties: lowest partition id) - the longest-first rule behind the 4/3 bound the paper cites (
 * DESIGN.md reading 3: the algorithm's body is missing from the paper's text).  Whole rows only (Observation 2,
 * PAPER.md:301-303).  This library does NOT shard this way (it splits heavy rows, reading 13); the
 * call exists to compare the two policies.
 *   deg_dev:  device int32 [dims[d]], scratch, receives the row degrees (computed on the device from the
 *             resident tensor copy; asynchronous work is synchronised before the host part runs).
 *   part_of_row: host int32 [dims[d]] or NULL, receives the partition of every row.
 *   loads:    host int64 [kappa], receives the nonzeros per partition.
 * Errors: EINVAL (null pointers, kappa < 1, d out of range), ECUDA.
 */
mttkrp_status_t mttkrp_partition_rows(mttkrp_handle_t h, int d, int kappa, int32_t* deg_dev /*device*/,
                                      int32_t* part_of_row /*host, may be NULL*/, int64_t* loads /*host*/,
                                      void* cuda_stream);

/* Library / build identification, e.g. "mttkrp_b200 0.1 sm_100a". */
const char* mttkrp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MTTKRP_B200_H */
