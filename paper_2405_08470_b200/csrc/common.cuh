// Internal declarations shared by the translation units of libmttkrp_b200 (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <vector>
#include "../../include/mttkrp.h"

namespace mk {

constexpr int kMaxModes = MTTKRP_MAX_MODES;
constexpr int kMaxShardNnz = 8192;   // nonzeros per thread-block shard (upper bound)
constexpr int kMinShardNnz = 1024;
constexpr int kMaxRank = 64;
constexpr int kBlockThreads = 256;   // MTTKRP kernel: 8 warps

void set_error(const char* fmt, ...);

#define MK_CUDA(call)                                                                        \
    do {                                                                                     \
        cudaError_t e__ = (call);                                                            \
        if (e__ != cudaSuccess) {                                                            \
            mk::set_error("%s:%d %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e__)); \
            return MTTKRP_ECUDA;                                                             \
        }                                                                                    \
    } while (0)

#define MK_TRY(expr)                              \
    do {                                          \
        mttkrp_status_t s__ = (expr);             \
        if (s__ != MTTKRP_OK) return s__;         \
    } while (0)

// Run-end flags.  A record of the mode-d layout is N uint32 key words (k_0 = i_d first) + the fp32
// value.  Indices are < 2^28, so bit 31 of a key word is free; the format builder and the remap pass
// store there, for the record at position j, e_l = "record j+1 differs from record j in one of the
// keys k_0..k_l" (the run of equal (k_0..k_l) ends at j): e_l sits in bit 31 of word l for
// 0 <= l <= N-2.  The last key word (the row gathered for every nonzero) carries no flag, so the hot
// loop turns it into an address with one multiply-add.  Padding records repeat the keys of the last
// nonzero (no run ends); the very last record of the padded array has every flag set.
constexpr uint32_t kFlag = 0x80000000u;
constexpr uint32_t kKeyMask = 0x0fffffffu;           // indices are < 2^28 (api.cu check_shape): bits 28..31 of a key word are free

// Cold-row marks (unpacked records, N <= 3).  The tensor is fixed, so which factor rows are re-used often is known
// before the first MTTKRP: mttkrp_create counts how often every index of a mode occurs (its degree) and calls a row
// COLD when it is not among the K most frequent rows of its factor matrix (K = MTTKRP_PREFETCH_ROWS, default 65536
// rows = 8 MB at R = 32; a factor with fewer rows has no cold row).  A gather of a cold row almost always misses L2
// when the factor matrices overflow it, and that miss decides how long the whole batch of gathers waits.  The
// record carries the mark for the row it gathers at the last level in bit 30 of key word 0 (word 0 is in a register
// in the hot loop anyway; the last key word itself stays flag-free) and, N = 3, for the row of its fiber level in
// bit 30 of key word 1.  The MTTKRP kernel requests marked rows into L2 one ring stage ahead (mttkrp_kernel.cu).
constexpr uint32_t kCold = 1u << 30;

// The flags are a property of (layout, position), so mttkrp_create computes them once per layout into a byte array
// and the record builder / remap pass only merges them into the key words.  Byte layout: bit l = e_l (l <= N-2); for
// N <= 3 also bit 6 = last-level row cold, bit 7 = fiber-level row cold.
template <int N>
__device__ __forceinline__ void apply_run_flags(uint32_t* k, uint32_t f) {
#pragma unroll
    for (int l = 0; l < N - 1; ++l) k[l] |= ((f >> l) & 1u) << 31;
    if constexpr (N <= 3) {
        k[0] |= ((f >> 6) & 1u) << 30;
        if constexpr (N == 3) k[1] |= ((f >> 7) & 1u) << 30;
    }
}

// Packed 16-byte records (N >= 4).  When the index widths allow, a record is {w0, w1, w2, val}: the keys of
// levels 0..N-2 are a bit string in the low bits of the 64-bit word (w1:w0) (level l at bit off[l], bits[l]
// wide), the N-1 run-end flags sit in its top bits (e_l at bit 63-l, i.e. bit 31-l of w1), and w2 is the last
// key, flag-free.  This is the paper's bit-level size accounting applied to the hot-path
// record: the remap then moves one 128-bit word per nonzero whatever N is.  Needs
// sum_{l<N-1} bits[l] + (N-1) <= 64 in every layout; otherwise the handle keeps 4*(N+1)-byte records.
struct PackDesc {
    int32_t bits[kMaxModes];
    int32_t off[kMaxModes];
};
__host__ __device__ __forceinline__ uint32_t pk_mask(int bits) { return bits >= 32 ? 0xffffffffu : ((1u << bits) - 1u); }
__device__ __forceinline__ uint32_t pk_get(uint32_t w0, uint32_t w1, int off, uint32_t mask) {
    return (uint32_t)(((((uint64_t)w1) << 32) | w0) >> off) & mask;
}
template <int N>
__device__ __forceinline__ uint4 pk_pack(const uint32_t* k, uint32_t flags, uint32_t val, const PackDesc& d) {
    uint64_t w01 = 0;
#pragma unroll
    for (int l = 0; l < N - 1; ++l) w01 |= ((uint64_t)k[l] << d.off[l]) | ((uint64_t)((flags >> l) & 1u) << (63 - l));
    return make_uint4((uint32_t)w01, (uint32_t)(w01 >> 32), k[N - 1], val);
}

// Field permutation of a remap pass: the key at level l of the destination layout is the key at level src[l] of
// the source layout.  RemapPk says where that source key sits in a packed record.
struct FieldMap { int src[kMaxModes]; };
struct RemapPk {
    int32_t soff[kMaxModes];      // bit offset of the source field in (w1:w0), or -1: it is w2 (the last key)
    uint32_t smask[kMaxModes];
};
// What the MTTKRP kernel needs to run Alg. 3 itself (Alg. 4 lines 15-19; MTTKRP_FUSE=1):
// T_out[scat[pos]] = the record at position pos, re-ordered for the next mode's layout.
struct FuseArgs {
    uint32_t* out_rec;            // T_out
    const uint32_t* scat;         // [nnz] remap id for mode (d+1) mod N: position in the next layout
    const uint8_t* sflags;        // [nnz] run-end flags of the next layout at that position
    int64_t nnz;                  // records beyond nnz are padding and are not scattered
    FieldMap fm;
    RemapPk rp;
    PackDesc dd;                  // packed records: bit layout of the next layout
};

// Test and experiment knobs (include/mttkrp.h, "Process environment variables").  The environment is read in ONE place,
// read_knobs (build.cu), by mttkrp_workspace_bytes and mttkrp_create before anything is launched; every value is
// checked there (a malformed one is MTTKRP_EINVAL, not a silent default) and the handle keeps the parsed copy.
struct Knobs {
    char key_order[16];           // MTTKRP_KEY_ORDER, "" = the library decides
    int pack;                     // MTTKRP_PACK: -1 unset / 0 / 1
    int remap_blocked;            // MTTKRP_REMAP_BLOCKED: -1 / 0 / 1
    int remap_block_log2;         // MTTKRP_REMAP_BLOCK_LOG2 clamped to [10,26], -1 unset
    int remap_twopass;            // MTTKRP_REMAP_TWOPASS: -1 / 0 / 1
    int twopass_window_log2;      // MTTKRP_TWOPASS_WINDOW_LOG2 clamped to [8,26], -1 unset
    int force_deep;               // MTTKRP_FORCE_DEEP: -1 / 0 / 1
    int64_t prefetch_rows;        // MTTKRP_PREFETCH_ROWS >= 0, -1 unset
    int fuse;                     // MTTKRP_FUSE: -1 / 0 / 1
    int policy;                   // MTTKRP_SHARD_POLICY: 0 equal (default), 1 alg1
    int kappa;                    // MTTKRP_KAPPA in [1,65536], 0 unset (one partition per SM)
};

// Per-mode tables built by mttkrp_create.
struct ModeMeta {
    int order[kMaxModes];     // sort-key order of this layout, order[0] == mode
    int pos[kMaxModes];       // pos[m] = level of mode m in `order`
    PackDesc pk;              // bit layout of this layout's packed records (handle->packed)
    uint32_t* next;           // [nnz] gather map of the remap d -> (d+1)%N: position in THIS layout of the
                              // element at position j of the next layout (the paper's remap id, read backwards)
    uint32_t* ord;            // (NULL after create when the chosen walk is the plain one)
                              // [nnz] positions of the NEXT layout ordered by the 2^block_log2-record block of this
                              // layout they come from (stable), or unused: the blocked remap walks the destination
                              // in this order so that its random reads stay inside one L2-resident window at a time
    uint32_t* osrc;           // [nnz] osrc[t] = next[ord[t]]: the source position of walk step t (saves the walk one
                              // dependent gather)
    int blocked;              // walk of the remap d -> (d+1)%N: 0 plain (destination order), 1 blocked (`ord`/`osrc`), 2 two
                              // passes (ord = scatter map into the window-grouped intermediate copy, osrc = gather map out of it)
    float plain_ms, twopass_ms;   // create-time measurements behind the choice of 2 (0 when not a candidate)
    int block_log2;
    double avg_run;           // average length of the ascending destination runs in `ord`
    uint8_t* lflags;          // [nnz_pad] run-end flags of THIS layout: bit l = e_l (see "Run-end flags")
    uint32_t* empty_rows;     // [n_empty] output rows without a nonzero
    int64_t n_empty;
    uint32_t* chains;         // [n_chains][3] = {first shard, last shard, row} for rows spanning shards
    int64_t n_chains;
    uint32_t* scat;           // MTTKRP_FUSE: [nnz] inverse of `next` (scatter form of the remap d -> (d+1)%N)
    uint8_t* sflags;          // MTTKRP_FUSE: [nnz] lflags of layout (d+1)%N read through scat
    uint32_t* bins;           // Alg. 1 policy: [kappa+1] first position of every partition in this layout
    int64_t max_bin, min_bin; // ... largest / smallest partition, in nonzeros
};

}  // namespace mk

namespace mk {
enum KernelClass { kClsRemap = 0, kClsZero = 1, kClsMttkrp = 2, kClsFixup = 3 };
struct TimedEvent { int cls; cudaEvent_t a, b; };
struct Timing {
    bool on = false;
    std::vector<TimedEvent> ev;
};
// Records an event pair around one launch when timing is on (RAII).
struct TimedLaunch {
    Timing* t; cudaStream_t st; TimedEvent e; bool active;
    TimedLaunch(Timing* timing, int cls, cudaStream_t s) : t(timing), st(s), active(false) {
        if (t && t->on) {
            e.cls = cls;
            if (cudaEventCreate(&e.a) == cudaSuccess && cudaEventCreate(&e.b) == cudaSuccess) {
                cudaEventRecord(e.a, st);
                active = true;
            }
        }
    }
    ~TimedLaunch() {
        if (active) { cudaEventRecord(e.b, st); t->ev.push_back(e); }
    }
};
}  // namespace mk

struct mttkrp_handle_s {
    int N;
    int64_t dims[mk::kMaxModes];
    int64_t nnz;
    int rec_words;            // N + 1 (N role-ordered int32 indices, then the fp32 value), or 4 when packed
    int packed;               // 1: 16-byte packed records (N >= 4 and the index widths fit, see PackDesc)
    int shard_nnz;
    int64_t num_shards;
    int fuse;                 // MTTKRP_FUSE=1: the MTTKRP kernel of mode d also writes the tensor copy of layout (d+1)%N
    int alt_layout;           // layout the OTHER tensor copy (rec_alt) holds completely, or -1
    int policy;               // 0: equal-nnz shards (default), 1: the paper's Alg. 1 (whole rows dealt to kappa partitions)
    int kappa;                // number of partitions of the Alg. 1 policy
    uint32_t* rec_cur;        // resident tensor copy T_in, layout `cur`
    uint32_t* rec_alt;        // T_out
    uint32_t* perm0;          // [nnz] original COO position of element k of layout 0
    mk::ModeMeta mode[mk::kMaxModes];
    float* carry;             // [2*num_shards][kMaxRank] partial rows of split rows
    int cur;
    uint32_t* jump[2];        // [nnz] each: composed gather maps for out-of-order calls (api.cu ensure_layout)
    const uint32_t* jump_map; // the cached composed map (points into jump[]) and the transition it serves
    int jump_from, jump_to;
    int max_rank;
    float* stage_fac[mk::kMaxModes];
    float* stage_out[mk::kMaxModes];
    int64_t bytes_held;
    int64_t remaps_done;
    int device;
    int num_sms;              // SM count of `device` (grid sizing)
    int force_deep;           // MTTKRP_FORCE_DEEP at create: -1 = by factor size (default), 0 / 1 = never / always
    mk::Knobs knobs;          // the environment as mttkrp_create read it
    uint32_t cold_deg[mk::kMaxModes];   // cold-row marks: a row of mode m is cold when its index occurs fewer than this many times (0: none)
    int64_t cold_rows[mk::kMaxModes];   // ... and how many rows of the mode that makes
    cudaStream_t last_stream; // stream of the last call that launched work for this handle
    cudaEvent_t ev_order;     // recorded on last_stream after every such call: a call on another stream waits on it
    int launched;             // ev_order has been recorded at least once
    mk::Timing* timing;       // owned; per-kernel event pairs while mttkrp_timing_begin is active
    cudaStream_t s_in, s_out; // copy streams of mttkrp_sweep_host (created on first use)
    cudaEvent_t ev_in[mk::kMaxModes], ev_done[mk::kMaxModes], ev_sync;
    int host_path_ready;
};

namespace mk {

// ---- build.cu -------------------------------------------------------------------------------
struct WorkspacePlan {
    size_t rec_a, rec_b, perm0, carry, jump[2];
    size_t next[kMaxModes], empty[kMaxModes], chains[kMaxModes], ord[kMaxModes], osrc[kMaxModes], lflags[kMaxModes], bins[kMaxModes], scat[kMaxModes], sflags[kMaxModes];
    size_t stage_fac[kMaxModes], stage_out[kMaxModes];
    size_t persistent_end;
    size_t scratch;          // start of the create-time scratch (may overlap rec_b)
    size_t pool, pool_slot;  // ord / osrc pool at the end of the workspace: 2*N slots of pool_slot bytes (ord[d], osrc[d])
    size_t total;
    int shard_nnz;
    int64_t num_shards;
};
// Host-side choice of the layouts (key order per mode) and of the record format; pure arithmetic on the shape.
struct LayoutPlan {
    int order[kMaxModes][kMaxModes];
    PackDesc pk[kMaxModes];
    int packed;
    int rec_words;
    int fuse;                // MTTKRP_FUSE=1 and 16-byte records and the default shard policy
    int policy;              // MTTKRP_SHARD_POLICY: 0 equal (default), 1 alg1
    int kappa;               // MTTKRP_KAPPA (alg1): 0 = one partition per SM
    Knobs knobs;             // every MTTKRP_* variable, parsed and checked
};
mttkrp_status_t read_knobs(Knobs* k);                                                    // EINVAL: malformed MTTKRP_* value
mttkrp_status_t plan_layouts(int N, const int64_t* dims, int64_t nnz, LayoutPlan* lp);   // EINVAL / EUNSUPPORTED: bad MTTKRP_* override
mttkrp_status_t plan_workspace(int N, const int64_t* dims, int64_t nnz, int max_rank, int rec_words, int num_sms, int kappa,
                               int fuse, WorkspacePlan* p);
// Alg. 1 (reading 3): rows by descending degree (ties: lower index), each to the least-loaded
// of kappa partitions (ties: lowest id).  Host code; returns false when out of memory.
bool lpt_partition(const int32_t* deg, int64_t rows, int kappa, int32_t* part_of_row, int64_t* loads);
int device_sm_count();       // SM count of the current device (148 when no device can be queried)
mttkrp_status_t build_format(mttkrp_handle_s* h, const WorkspacePlan& plan, char* ws,
                             const int32_t* idx, const float* vals, cudaStream_t st);

// ---- remap.cu -------------------------------------------------------------------------------
mttkrp_status_t launch_remap(mttkrp_handle_s* h, int from, int to, const uint32_t* jump, cudaStream_t st);   // swaps copies
constexpr int kTwoPassWindowLog2 = 21;      // destination window of the two-pass remap: 2^21 records (32 MB), L2-resident
void remap_fields(const mttkrp_handle_s* h, int from, int to, FieldMap* fm, RemapPk* rp);
mttkrp_status_t launch_remap_padding(mttkrp_handle_s* h, int from, int to, cudaStream_t st);   // padding records of rec_alt only
mttkrp_status_t launch_export(const mttkrp_handle_s* h, int32_t* idx, float* vals, cudaStream_t st);
mttkrp_status_t launch_row_degrees(const mttkrp_handle_s* h, int d, int32_t* deg_dev, cudaStream_t st);
mttkrp_status_t launch_perm_step(const uint32_t* map, const uint32_t* in, uint32_t* out, int64_t nnz, cudaStream_t st);

// ---- mttkrp_kernel.cu -----------------------------------------------------------------------
mttkrp_status_t launch_mttkrp(mttkrp_handle_s* h, int d, const float* const* factors, int R,
                              float* out, cudaStream_t st);

}  // namespace mk
