// On-device format builder (mttkrp_create): hand-written stable LSD radix sort of the nonzeros by
// each mode's key tuple, position maps between consecutive layouts (the paper's remap ids,
// PAPER.md:185; unique per element, Observation 1 PAPER.md:297-299), the mode-0 tensor copy
// (PAPER.md:145), and per-mode tables (empty output rows; rows that span shards).
// The paper builds its format on the CPU (Sec. 5.7); here it is done on the GPU.
#include <cerrno>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <functional>
#include <new>
#include <queue>
#include <utility>
#include <vector>
#include "common.cuh"

namespace mk {

// ----------------------------------------------------------------------------------------------
// workspace plan
// ----------------------------------------------------------------------------------------------
static inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

constexpr int kSortThreads = 256;
constexpr int kSortItems = 16;
constexpr int kSortTile = kSortThreads * kSortItems;   // keys per block per radix pass
constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanThreads * kScanItems;
constexpr int kDegBins = 1024;                          // bins of the degree histogram behind the cold-row marks (deg_bin)

int device_sm_count() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) {
        (void)cudaGetLastError();
        return 148;                                   // B200; only reached without a device (size queries on a CPU box)
    }
    return sms;
}

static int choose_shard_nnz(int64_t nnz, int num_sms) {
    // Aim for >= 8 shards per SM; power of two in [kMinShardNnz, kMaxShardNnz].
    int s = kMaxShardNnz;
    while (s > kMinShardNnz && nnz / s < (int64_t)num_sms * 8) s >>= 1;
    return s;
}

mttkrp_status_t plan_workspace(int N, const int64_t* dims, int64_t nnz, int max_rank, int rec_words, int num_sms,
                               int kappa, int fuse, WorkspacePlan* p) {
    memset(p, 0, sizeof(*p));
    const size_t n = (size_t)nnz;
    p->shard_nnz = choose_shard_nnz(nnz, num_sms);
    p->num_shards = (nnz + p->shard_nnz - 1) / p->shard_nnz;
    // both tensor copies are padded to a whole number of shards (zero-valued copies of the last nonzero)
    const size_t rec_bytes = (size_t)rec_words * 4 * (size_t)(p->num_shards * p->shard_nnz);
    size_t off = 0;
    p->rec_a = off; off = align_up(off + rec_bytes);
    for (int d = 0; d < N; ++d) { p->next[d] = off; off = align_up(off + 4 * n); }
    for (int d = 0; d < N; ++d) { p->lflags[d] = off; off = align_up(off + (size_t)(p->num_shards * p->shard_nnz)); }
    p->perm0 = off; off = align_up(off + 4 * n);
    // composed maps for out-of-order calls: a jump of k layouts composes k-1 times (ping-pong when k > 2)
    p->jump[0] = off; if (N >= 3) off = align_up(off + 4 * n);
    p->jump[1] = off; if (N >= 4) off = align_up(off + 4 * n);
    for (int d = 0; d < N; ++d) { p->empty[d] = off; off = align_up(off + 4 * (size_t)dims[d]); }
    for (int d = 0; d < N; ++d) { p->chains[d] = off; off = align_up(off + 12 * (size_t)p->num_shards); }
    for (int d = 0; d < N; ++d) { p->bins[d] = off; if (kappa > 0) off = align_up(off + 4 * ((size_t)kappa + 1)); }
    for (int d = 0; d < N; ++d) { p->scat[d] = off; if (fuse) off = align_up(off + 4 * n); }
    for (int d = 0; d < N; ++d) { p->sflags[d] = off; if (fuse) off = align_up(off + n); }
    p->carry = off; off = align_up(off + (size_t)2 * p->num_shards * kMaxRank * 4);
    if (max_rank > 0) {
        for (int d = 0; d < N; ++d) { p->stage_fac[d] = off; off = align_up(off + (size_t)dims[d] * max_rank * 4); }
        for (int d = 0; d < N; ++d) { p->stage_out[d] = off; off = align_up(off + (size_t)dims[d] * max_rank * 4); }
    }
    p->persistent_end = off;
    p->rec_b = off;
    p->scratch = off;
    int64_t maxdim = 1;
    for (int d = 0; d < N; ++d) maxdim = std::max<int64_t>(maxdim, dims[d]);
    const size_t nblocks = (n + kSortTile - 1) / kSortTile;
    size_t scratch = 0;
    scratch += 4 * align_up(4 * n);                                   // key/perm ping-pong
    scratch += align_up(4 * (256 * nblocks + 1));                     // digit histogram table
    scratch += 2 * align_up(4 * ((size_t)std::max<int64_t>(maxdim, p->num_shards) + 1));   // flags + positions
    scratch += align_up(4 * (std::max<size_t>(256 * nblocks + 1, (size_t)maxdim + 1) / kScanTile + 2));  // scan block sums
    scratch += 4096;                                                  // counters, error flag
    for (int d = 0; d < N; ++d) scratch += align_up(4 * ((size_t)dims[d] + 1));   // index degrees (cold-row marks)
    scratch += align_up(4 * kDegBins);                                // degree histogram
    // ord / osrc (8 bytes per nonzero per transition) sit in a pool at the very END of the workspace: which
    // transitions need them is only known once create has measured the walks, and those that do are then moved to the
    // front of the pool (build_format), so that everything the handle still uses afterwards is one prefix of the
    // workspace (info.bytes_held) and the rest is the caller's again.
    p->pool = off + std::max(align_up(rec_bytes), scratch);
    p->pool_slot = align_up(4 * n);
    for (int d = 0; d < N; ++d) {
        p->ord[d] = p->pool + (size_t)(2 * d) * p->pool_slot;
        p->osrc[d] = p->pool + (size_t)(2 * d + 1) * p->pool_slot;
    }
    p->total = p->pool + (size_t)(2 * N) * p->pool_slot;
    return MTTKRP_OK;
}

// ----------------------------------------------------------------------------------------------
// small kernels
// ----------------------------------------------------------------------------------------------
__global__ void k_validate(const int32_t* __restrict__ idx, int64_t nnz, int N, const int64_t* __restrict__ dims_dev,
                           uint32_t* __restrict__ bad) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int m = blockIdx.y;
    if (k < nnz) {
        int32_t v = idx[(size_t)m * nnz + k];
        if (v < 0 || (int64_t)v >= dims_dev[m]) atomicOr(bad, 1u << m);
    }
}

// deg[key[k]] += 1 (Alg. 1's vertex degrees; create time only, global atomics are fine here)
__global__ void k_count_keys(const uint32_t* __restrict__ key, int64_t n, uint32_t* __restrict__ deg) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) atomicAdd(deg + key[k], 1u);
}

// Same count with the lanes of a warp that hit the same key combined first (Zipf-skewed modes put a fifth of the
// nonzeros on one counter).
__global__ void k_count_keys_agg(const uint32_t* __restrict__ key, int64_t n, uint32_t* __restrict__ deg) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool in = k < n;
    const uint32_t v = in ? key[k] : 0xffffffffu;
    const unsigned peers = __match_any_sync(0xffffffffu, v);
    if (in && (int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(deg + v, (uint32_t)__popc(peers));
}

// Degree histogram on a log-linear scale (exact below 64, then 32 steps per octave): the host reads it to turn
// "the K most frequent rows" into a degree threshold (cold-row marks, common.cuh).
__host__ __device__ inline int deg_bin(uint32_t deg) {
    if (deg < 64u) return (int)deg;
    int lg = 31;
    while (!((deg >> lg) & 1u)) --lg;                   // floor(log2 deg) >= 6
    return 64 + (lg - 6) * 32 + (int)((deg >> (lg - 5)) & 31u);
}
__host__ __device__ inline uint32_t deg_bin_floor(int bin) {      // smallest degree that falls into `bin`
    if (bin < 64) return (uint32_t)bin;
    const int lg = (bin - 64) / 32 + 6, sub = (bin - 64) % 32;
    return (uint32_t)(32 + sub) << (lg - 5);
}
__global__ void k_degree_hist(const uint32_t* __restrict__ deg, int64_t rows, uint32_t* __restrict__ hist) {
    __shared__ uint32_t h[kDegBins];
    for (int i = threadIdx.x; i < kDegBins; i += blockDim.x) h[i] = 0;
    __syncthreads();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < rows; i += (int64_t)gridDim.x * blockDim.x)
        atomicAdd(&h[deg_bin(deg[i])], 1u);
    __syncthreads();
    for (int i = threadIdx.x; i < kDegBins; i += blockDim.x)
        if (h[i]) atomicAdd(hist + i, h[i]);
}

__global__ void k_iota(uint32_t* __restrict__ p, int64_t n) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) p[k] = (uint32_t)k;
}

// key[k] = col[perm[k]]
__global__ void k_gather_u32(const uint32_t* __restrict__ col, const uint32_t* __restrict__ perm,
                             uint32_t* __restrict__ key, int64_t n) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) key[k] = col[perm[k]];
}

// p[k] = table[p[k]] (in place)
__global__ void k_apply_table(const uint32_t* __restrict__ table, uint32_t* p, int64_t n) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) p[k] = table[p[k]];
}

// inv[perm[j]] = j
__global__ void k_invert(const uint32_t* __restrict__ perm, uint32_t* __restrict__ inv, int64_t n) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) inv[perm[j]] = (uint32_t)j;
}

// ----------------------------------------------------------------------------------------------
// exclusive scan (uint32), three phases; in and out may alias
// ----------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total, uint32_t* smem /*>=33*/) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) smem[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = (lane < (int)(blockDim.x >> 5)) ? smem[lane] : 0;
        uint32_t winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        smem[lane] = winc - w;
        if (lane == 31) smem[32] = winc;
    }
    __syncthreads();
    uint32_t res = smem[warp] + inc - v;
    *total = smem[32];
    __syncthreads();
    return res;
}

__global__ void __launch_bounds__(kScanThreads) k_scan_reduce(const uint32_t* __restrict__ in, int64_t n,
                                                              uint32_t* __restrict__ sums) {
    __shared__ uint32_t sm[33];
    int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i)
        if (base + i < n) s += in[base + i];
    uint32_t tot;
    block_exclusive_scan(s, &tot, sm);
    if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(1024) k_scan_sums(uint32_t* __restrict__ sums, int64_t nb) {
    __shared__ uint32_t sm[33];
    uint32_t carry = 0;
    for (int64_t base = 0; base < nb; base += 1024) {
        int64_t i = base + threadIdx.x;
        uint32_t v = (i < nb) ? sums[i] : 0;
        uint32_t tot;
        uint32_t ex = block_exclusive_scan(v, &tot, sm);
        if (i < nb) sums[i] = carry + ex;
        carry += tot;
    }
}

__global__ void __launch_bounds__(kScanThreads) k_scan_apply(const uint32_t* in, uint32_t* out, int64_t n,
                                                             const uint32_t* __restrict__ sums) {
    __shared__ uint32_t sm[33];
    int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    uint32_t v[kScanItems];
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        v[i] = (base + i < n) ? in[base + i] : 0;
        s += v[i];
    }
    uint32_t tot;
    uint32_t ex = block_exclusive_scan(s, &tot, sm) + sums[blockIdx.x];
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (base + i < n) out[base + i] = ex;
        ex += v[i];
    }
}

static mttkrp_status_t exclusive_scan(uint32_t* data, int64_t n, uint32_t* sums, cudaStream_t st) {
    if (n <= 0) return MTTKRP_OK;
    int64_t nb = (n + kScanTile - 1) / kScanTile;
    k_scan_reduce<<<(unsigned)nb, kScanThreads, 0, st>>>(data, n, sums);
    k_scan_sums<<<1, 1024, 0, st>>>(sums, nb);
    k_scan_apply<<<(unsigned)nb, kScanThreads, 0, st>>>(data, data, n, sums);
    MK_CUDA(cudaGetLastError());
    return MTTKRP_OK;
}

// ----------------------------------------------------------------------------------------------
// stable LSD radix pass over (key, payload) pairs, 8-bit digits
// ----------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kSortThreads) k_radix_hist(const uint32_t* __restrict__ keys, int64_t n, int shift,
                                                             uint32_t* __restrict__ hist, int64_t nblocks) {
    __shared__ uint32_t cnt[256];
    cnt[threadIdx.x] = 0;
    __syncthreads();
    int64_t base = (int64_t)blockIdx.x * kSortTile;
#pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
        int64_t k = base + (int64_t)i * kSortThreads + threadIdx.x;
        if (k < n) atomicAdd(&cnt[(keys[k] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * nblocks + blockIdx.x] = cnt[threadIdx.x];
}

// Block b owns keys [b*tile, (b+1)*tile); warp w owns a contiguous 32*items slice of it, item i of
// lane l being element slice + i*32 + l.  Ranks are assigned in exactly that memory order, so equal
// digits keep their input order (stability).
__global__ void __launch_bounds__(kSortThreads) k_radix_scatter(const uint32_t* __restrict__ keys_in,
                                                                const uint32_t* __restrict__ vals_in,
                                                                uint32_t* __restrict__ keys_out,
                                                                uint32_t* __restrict__ vals_out, int64_t n, int shift,
                                                                const uint32_t* __restrict__ offs, int64_t nblocks) {
    constexpr int kWarps = kSortThreads / 32;
    __shared__ uint32_t cnt[kWarps][256];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < kWarps * 256; i += kSortThreads) (&cnt[0][0])[i] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * kSortTile + (int64_t)warp * (32 * kSortItems);
    uint32_t key[kSortItems], val[kSortItems], rnk[kSortItems];
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
        int64_t k = base + i * 32 + lane;
        bool valid = k < n;
        key[i] = valid ? keys_in[k] : 0u;
        val[i] = valid ? vals_in[k] : 0u;
        unsigned dig = valid ? ((key[i] >> shift) & 255u) : 256u;
        unsigned peers = __match_any_sync(0xffffffffu, dig);
        unsigned before = __popc(peers & lt);
        uint32_t old = 0;
        if (valid) old = cnt[warp][dig];
        __syncwarp();
        if (valid && before == 0) cnt[warp][dig] = old + __popc(peers);
        __syncwarp();
        rnk[i] = old + before;
    }
    __syncthreads();
    {
        const int dig = threadIdx.x;   // kSortThreads == 256 digits
        uint32_t run = offs[(size_t)dig * nblocks + blockIdx.x];
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            uint32_t c = cnt[w][dig];
            cnt[w][dig] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
        int64_t k = base + i * 32 + lane;
        if (k < n) {
            unsigned dig = (key[i] >> shift) & 255u;
            uint32_t pos = cnt[warp][dig] + rnk[i];
            keys_out[pos] = key[i];
            vals_out[pos] = val[i];
        }
    }
}

// ----------------------------------------------------------------------------------------------
// records, maps, tables
// ----------------------------------------------------------------------------------------------
// rec[k] = { idx[order[0]][perm[k]], ..., idx[order[N-1]][perm[k]], val[perm[k]] }
struct OrderArg { int v[kMaxModes]; };

// Run-end flags of one layout (common.cuh): bit l of flags[k] = e_l = "the record at k+1 differs from
// the record at k in one of the keys k_0..k_l".  Padding positions repeat the last nonzero (no run
// ends); the last position of the padded array has every flag set.
// For N <= 3 the byte also carries the cold-row marks (common.cuh): bit 6 = the last-level row, bit 7 = the fiber-level
// row (N = 3) is cold, i.e. its index occurs fewer than cold.t[c] times in the tensor.  cold.deg[c] == nullptr: no marks.
struct ColdArg {
    const uint32_t* deg[2];
    uint32_t t[2];
};
__global__ void k_build_flags(const int32_t* __restrict__ idx, const uint32_t* __restrict__ perm, int64_t nnz,
                              int64_t nnz_pad, int N, OrderArg order, ColdArg cold, uint8_t* __restrict__ flags) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nnz_pad) return;
    const bool last = k + 1 >= nnz_pad;
    const uint32_t src = perm[k < nnz ? k : nnz - 1];
    const uint32_t nsrc = last ? src : perm[k + 1 < nnz ? k + 1 : nnz - 1];
    bool diff = last;
    uint32_t f = 0;
    for (int l = 0; l < N - 1; ++l) {
        const size_t col = (size_t)order.v[l] * nnz;
        diff = diff || (idx[col + src] != idx[col + nsrc]);
        f |= (diff ? 1u : 0u) << l;
    }
    if (N <= 3) {
        for (int c = 0; c < N - 1; ++c) {                // c = 0: last level (key N-1), c = 1: fiber level (key N-2)
            if (!cold.deg[c]) continue;
            const uint32_t dg = cold.deg[c][idx[(size_t)order.v[N - 1 - c] * nnz + src]];
            f |= (dg < cold.t[c] ? 1u : 0u) << (6 + c);
        }
    }
    flags[k] = (uint8_t)f;
}

// rec[k] = keys of the nonzero perm[k] in the layout's key order (with its run-end flags merged into
// bit 31, common.cuh) + value.  Positions k in [nnz, nnz_pad) are padding: the keys of the last
// nonzero with value 0.
__global__ void k_build_records(const int32_t* __restrict__ idx, const float* __restrict__ vals,
                                const uint32_t* __restrict__ perm, const uint8_t* __restrict__ flags, int64_t nnz,
                                int64_t nnz_pad, int N, OrderArg order, uint32_t* __restrict__ rec) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nnz_pad) return;
    const uint32_t src = perm[k < nnz ? k : nnz - 1];
    const uint32_t f = flags[k];
    uint32_t* r = rec + (size_t)k * (N + 1);
    for (int l = 0; l < N; ++l) {
        uint32_t key = (uint32_t)idx[(size_t)order.v[l] * nnz + src];
        if (l <= N - 2) key |= ((f >> l) & 1u) << 31;                  // e_l rides on key word l (common.cuh)
        if (N <= 3 && l == 0) key |= ((f >> 6) & 1u) << 30;             // cold-row mark of the last-level row
        if (N == 3 && l == 1) key |= ((f >> 7) & 1u) << 30;             // ... of the fiber-level row
        r[l] = key;
    }
    r[N] = k < nnz ? __float_as_uint(vals[src]) : 0u;
}

// Packed variant (common.cuh PackDesc): one 16-byte record per nonzero.
template <int N>
__global__ void k_build_records_pk(const int32_t* __restrict__ idx, const float* __restrict__ vals,
                                   const uint32_t* __restrict__ perm, const uint8_t* __restrict__ flags, int64_t nnz,
                                   int64_t nnz_pad, OrderArg order, PackDesc pd, uint4* __restrict__ rec) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nnz_pad) return;
    const uint32_t src = perm[k < nnz ? k : nnz - 1];
    uint32_t key[N];
#pragma unroll
    for (int l = 0; l < N; ++l) key[l] = (uint32_t)idx[(size_t)order.v[l] * nnz + src];
    rec[k] = pk_pack<N>(key, flags[k], k < nnz ? __float_as_uint(vals[src]) : 0u, pd);
}

// out[k] = table[idx[k]] for byte tables
__global__ void k_gather_u8(const uint8_t* __restrict__ table, const uint32_t* __restrict__ idx, uint8_t* __restrict__ out, int64_t n) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) out[k] = table[idx[k]];
}

// out[b[a[m]]] = m
__global__ void k_invert_through(const uint32_t* __restrict__ a, const uint32_t* __restrict__ b, uint32_t* __restrict__ out, int64_t n) {
    int64_t m = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (m < n) out[b[a[m]]] = (uint32_t)m;
}

// key[j] = map[j] >> shift (the source block of destination position j)
__global__ void k_block_keys(const uint32_t* __restrict__ map, int shift, uint32_t* __restrict__ key, int64_t n) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) key[j] = map[j] >> shift;
}

// counts the positions t with ord[t+1] != ord[t] + 1 (run breaks)
__global__ void k_count_breaks(const uint32_t* __restrict__ ord, int64_t n, uint32_t* __restrict__ counter) {
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool brk = (t + 1 < n) && (ord[t + 1] != ord[t] + 1u);
    const unsigned m = __ballot_sync(0xffffffffu, brk);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(counter, (uint32_t)__popc(m));
}

__global__ void k_mark_rows(const uint32_t* __restrict__ kd, int64_t nnz, uint32_t* __restrict__ present) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < nnz) present[kd[k]] = 1u;
}

// flags[i] = 1 - present[i] for i < rows, flags[rows] = 0
__global__ void k_invert_flags(uint32_t* __restrict__ flags, int64_t rows) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < rows) flags[i] = 1u - flags[i];
    else if (i == rows) flags[i] = 0u;
}

// After the exclusive scan pos[] of the flags: compact the flagged ids.  A flagged id i has
// pos[i+1] == pos[i] + 1.
__global__ void k_compact_ids(const uint32_t* __restrict__ pos, int64_t n, uint32_t* __restrict__ list) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && pos[i + 1] != pos[i]) list[pos[i]] = (uint32_t)i;
}

// Shard s covers positions [s*S, min((s+1)*S, nnz)).  A chain starts at s when the last row of s
// continues into s+1 and that row begins inside s.
__global__ void k_chain_flags(const uint32_t* __restrict__ kd, int64_t nnz, int S, int64_t nshards,
                              uint32_t* __restrict__ flags) {
    int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s > nshards) return;
    if (s == nshards) { flags[s] = 0; return; }
    int64_t end = min((s + 1) * (int64_t)S, nnz);
    uint32_t f = 0;
    if (end < nnz) {
        uint32_t r = kd[end - 1];
        if (kd[end] == r) f = (s == 0 || kd[s * (int64_t)S - 1] != r) ? 1u : 0u;
    }
    flags[s] = f;
}

__global__ void k_chain_fill(const uint32_t* __restrict__ kd, int64_t nnz, int S, int64_t nshards,
                             const uint32_t* __restrict__ pos, uint32_t* __restrict__ chains) {
    int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nshards || pos[s + 1] == pos[s]) return;
    int64_t end = min((s + 1) * (int64_t)S, nnz);
    uint32_t r = kd[end - 1];
    // upper bound of r in kd[end, nnz)
    int64_t lo = end, hi = nnz;
    while (lo < hi) {
        int64_t mid = (lo + hi) >> 1;
        if (kd[mid] <= r) lo = mid + 1; else hi = mid;
    }
    uint32_t* c = chains + (size_t)pos[s] * 3;
    c[0] = (uint32_t)s;
    c[1] = (uint32_t)((lo - 1) / S);
    c[2] = r;
}

bool lpt_partition(const int32_t* deg, int64_t rows, int kappa, int32_t* part_of_row, int64_t* loads) {
    try {
        std::vector<int32_t> order((size_t)rows);
        for (int64_t i = 0; i < rows; ++i) order[(size_t)i] = (int32_t)i;
        std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return deg[a] > deg[b]; });
        typedef std::pair<int64_t, int> Bin;                   // (load, partition id): min-heap, ties to the lowest id
        std::priority_queue<Bin, std::vector<Bin>, std::greater<Bin>> heap;
        for (int z = 0; z < kappa; ++z) { loads[z] = 0; heap.push(Bin(0, z)); }
        for (int64_t q = 0; q < rows; ++q) {
            const int32_t v = order[(size_t)q];
            Bin b = heap.top();
            heap.pop();
            b.first += deg[v];
            loads[b.second] = b.first;
            if (part_of_row) part_of_row[v] = b.second;
            heap.push(b);
        }
    } catch (...) {
        return false;
    }
    return true;
}

static inline unsigned grid_for(int64_t n, int threads) { return (unsigned)std::max<int64_t>(1, (n + threads - 1) / threads); }

static int ceil_log2_i64(int64_t x) {
    int b = 0;
    while (((int64_t)1 << b) < x) ++b;
    return b;
}

static bool known_key_order(const char* s) {
    return !strcmp(s, "revcyclic") || !strcmp(s, "desc") || !strcmp(s, "asc") || !strcmp(s, "cyclic");
}

void choose_key_order(int N, const int64_t* dims, int d, const char* env, int* order) {
    // Default: order[d] = (d, d-1, d-2, ..., d-N+1) (mod N).  The layout of mode d+1 is then
    // (last key of layout d, then the keys of layout d in their order), so inside one output row of
    // mode d+1 the nonzeros appear in the same order as in layout d: the remap d -> d+1 is a stable
    // partition by a single key, and the nonzeros that a block of layout d sends to one output row
    // stay contiguous (what the blocked remap needs, remap.cu).  DESIGN.md reading 4.
    // `env` (mttkrp_create: MTTKRP_KEY_ORDER, or "desc" when the modes are too large for the blocked
    // remap to pay) selects other tuples: desc / asc = the other modes by size, cyclic = d+1, d+2, ...
    order[0] = d;
    if (!env || strcmp(env, "revcyclic") == 0) {
        for (int j = 1; j < N; ++j) order[j] = ((d - j) % N + N) % N;
        return;
    }
    int rest[kMaxModes], n = 0;
    for (int j = 1; j < N; ++j) rest[n++] = (d + j) % N;     // cyclic
    if (strcmp(env, "cyclic") != 0) {
        bool asc = strcmp(env, "asc") == 0;
        std::sort(rest, rest + n, [&](int a, int b) {
            if (dims[a] != dims[b]) return asc ? dims[a] < dims[b] : dims[a] > dims[b];
            return a < b;
        });
    }
    for (int j = 0; j < n; ++j) order[j + 1] = rest[j];
}

// ---- environment knobs ---------------------------------------------------------------------------------------
// 0/1 switches accept exactly "0" or "1"; integers must be decimal numbers with nothing after them.
static mttkrp_status_t env_flag(const char* name, int* out) {
    *out = -1;
    const char* e = getenv(name);
    if (!e) return MTTKRP_OK;
    if ((e[0] == '0' || e[0] == '1') && e[1] == '\0') { *out = e[0] - '0'; return MTTKRP_OK; }
    set_error("%s=%s is not 0 or 1", name, e);
    return MTTKRP_EINVAL;
}
static mttkrp_status_t env_int(const char* name, long long lo, long long hi, bool clamp, long long unset, long long* out) {
    *out = unset;
    const char* e = getenv(name);
    if (!e) return MTTKRP_OK;
    char* end = nullptr;
    errno = 0;
    const long long v = strtoll(e, &end, 10);
    if (end == e || *end != '\0' || errno != 0) { set_error("%s=%s is not an integer", name, e); return MTTKRP_EINVAL; }
    if (v < lo || v > hi) {
        if (!clamp) { set_error("%s=%s outside [%lld, %lld]", name, e, lo, hi); return MTTKRP_EINVAL; }
        *out = v < lo ? lo : hi;
        return MTTKRP_OK;
    }
    *out = v;
    return MTTKRP_OK;
}

mttkrp_status_t read_knobs(Knobs* k) {
    memset(k, 0, sizeof(*k));
    if (const char* e = getenv("MTTKRP_KEY_ORDER")) {
        if (!known_key_order(e)) { set_error("MTTKRP_KEY_ORDER=%s is not one of revcyclic, desc, asc, cyclic", e); return MTTKRP_EINVAL; }
        snprintf(k->key_order, sizeof(k->key_order), "%s", e);
    }
    long long v = 0;
    MK_TRY(env_flag("MTTKRP_PACK", &k->pack));                       // 0 forces 4*(N+1)-byte records (tests)
    MK_TRY(env_flag("MTTKRP_REMAP_BLOCKED", &k->remap_blocked));     // 0 / 1 force the walk (experiments)
    MK_TRY(env_flag("MTTKRP_REMAP_TWOPASS", &k->remap_twopass));     // 0 / 1 force the walk (tests, experiments)
    MK_TRY(env_flag("MTTKRP_FORCE_DEEP", &k->force_deep));           // 0 / 1 pins the kernel variant (tests)
    MK_TRY(env_flag("MTTKRP_FUSE", &k->fuse));                       // 1: Alg. 3 runs inside the MTTKRP kernel
    MK_TRY(env_int("MTTKRP_REMAP_BLOCK_LOG2", 10, 26, true, -1, &v));    k->remap_block_log2 = (int)v;
    MK_TRY(env_int("MTTKRP_TWOPASS_WINDOW_LOG2", 8, 26, true, -1, &v));  k->twopass_window_log2 = (int)v;
    MK_TRY(env_int("MTTKRP_PREFETCH_ROWS", 0, (1ll << 40), false, -1, &v)); k->prefetch_rows = v;
    MK_TRY(env_int("MTTKRP_KAPPA", 1, 65536, false, 0, &v));             k->kappa = (int)v;
    if (const char* pol = getenv("MTTKRP_SHARD_POLICY")) {           // equal (default) | alg1 (the paper's partitioner)
        if (strcmp(pol, "equal") != 0 && strcmp(pol, "alg1") != 0) {
            set_error("MTTKRP_SHARD_POLICY=%s is not one of equal, alg1", pol);
            return MTTKRP_EINVAL;
        }
        k->policy = strcmp(pol, "alg1") == 0 ? 1 : 0;
    }
    return MTTKRP_OK;
}

mttkrp_status_t plan_layouts(int N, const int64_t* dims, int64_t nnz, LayoutPlan* lp) {
    memset(lp, 0, sizeof(*lp));
    MK_TRY(read_knobs(&lp->knobs));
    const Knobs& kn = lp->knobs;
    // Key order of the layouts (reading 4).  The default makes every remap a stable partition
    // by one key, which the blocked remap turns into L2-resident gathers; that pays when the nonzeros a
    // source block sends to one output row form runs of several records.  The expected run for mode d
    // is nnz / (dims[d] * number of blocks); when most modes are too large for that, the size-ordered
    // tuple (one remap of the cycle moves whole fibers) is the better choice.
    const char* order_env = kn.key_order[0] ? kn.key_order : nullptr;
    if (!order_env) {
        const double nblk = (double)((nnz >> 20) > 0 ? (nnz >> 20) : 1);
        int good = 0;
        for (int d = 0; d < N; ++d) good += ((double)nnz / ((double)dims[d] * nblk) >= 1.0) ? 1 : 0;
        order_env = (2 * good >= N) ? "revcyclic" : "desc";
    }
    for (int d = 0; d < N; ++d) choose_key_order(N, dims, d, order_env, lp->order[d]);
    // Record format: packed 16-byte records for N >= 4 when every layout fits (common.cuh PackDesc).
    bool packed = N >= 4 && kn.pack != 0;
    for (int d = 0; d < N && packed; ++d) {
        int off = 0;
        for (int l = 0; l < N; ++l) {
            const int b = std::max(1, ceil_log2_i64(dims[lp->order[d][l]]));
            lp->pk[d].bits[l] = b;
            lp->pk[d].off[l] = (l < N - 1) ? off : 0;
            if (l < N - 1) off += b;
        }
        if (off + (N - 1) > 64) packed = false;                       // keys of levels 0..N-2 + N-1 flags in 64 bits
    }
    lp->packed = packed ? 1 : 0;
    lp->rec_words = packed ? 4 : N + 1;
    lp->policy = kn.policy;
    lp->kappa = kn.kappa;
    // The fused kernel exists for 16-byte records under the default shard policy; asking for it where it cannot
    // run is an error the caller sees, not a request that is dropped.
    lp->fuse = 0;
    if (kn.fuse == 1) {
        if (lp->rec_words != 4) {
            set_error("MTTKRP_FUSE=1 needs 16-byte records (nmodes == 3, or nmodes >= 4 with packed records); this tensor has %d-byte records",
                      4 * lp->rec_words);
            return MTTKRP_EUNSUPPORTED;
        }
        if (lp->policy != 0) { set_error("MTTKRP_FUSE=1 cannot be combined with MTTKRP_SHARD_POLICY=alg1"); return MTTKRP_EUNSUPPORTED; }
        lp->fuse = 1;
    }
    return MTTKRP_OK;
}

mttkrp_status_t build_format(mttkrp_handle_s* h, const WorkspacePlan& plan, char* ws, const int32_t* idx,
                             const float* vals, cudaStream_t st) {
    const int N = h->N;
    const int64_t nnz = h->nnz;
    const size_t n = (size_t)nnz;
    const int S = h->shard_nnz;
    const int64_t nshards = h->num_shards;
    int64_t maxdim = 1;
    for (int d = 0; d < N; ++d) maxdim = std::max<int64_t>(maxdim, h->dims[d]);
    const int64_t nblocks = (nnz + kSortTile - 1) / kSortTile;

    // scratch carve-up (mirrors plan_workspace)
    char* sp = ws + plan.scratch;
    auto take = [&](size_t bytes) { char* p = sp; sp += align_up(bytes); return p; };
    uint32_t* keyA = (uint32_t*)take(4 * n);
    uint32_t* keyB = (uint32_t*)take(4 * n);
    uint32_t* permA = (uint32_t*)take(4 * n);
    uint32_t* permB = (uint32_t*)take(4 * n);
    uint32_t* hist = (uint32_t*)take(4 * (256 * (size_t)nblocks + 1));
    const size_t flag_n = (size_t)std::max<int64_t>(maxdim, nshards) + 1;
    uint32_t* flags = (uint32_t*)take(4 * flag_n);
    uint32_t* flags2 = (uint32_t*)take(4 * flag_n);
    uint32_t* sums = (uint32_t*)take(4 * (std::max<size_t>(256 * (size_t)nblocks + 1, (size_t)maxdim + 1) / kScanTile + 2));
    uint32_t* small = (uint32_t*)take(4096);          // [0]=bad flag, [8..8+2N) counts, then dims
    int64_t* dims_dev = (int64_t*)(small + 64);
    uint32_t* degs[kMaxModes];
    for (int d = 0; d < N; ++d) degs[d] = (uint32_t*)take(4 * ((size_t)h->dims[d] + 1));
    uint32_t* dhist = (uint32_t*)take(4 * kDegBins);

    MK_CUDA(cudaMemsetAsync(small, 0, 4096, st));
    MK_CUDA(cudaMemcpyAsync(dims_dev, h->dims, sizeof(int64_t) * N, cudaMemcpyHostToDevice, st));

    if (nnz > 0) {
        dim3 g(grid_for(nnz, 256), N);
        k_validate<<<g, 256, 0, st>>>(idx, nnz, N, dims_dev, small);
        MK_CUDA(cudaGetLastError());
        uint32_t bad = 0;
        MK_CUDA(cudaMemcpyAsync(&bad, small, 4, cudaMemcpyDeviceToHost, st));
        MK_CUDA(cudaStreamSynchronize(st));
        if (bad) {
            set_error("index out of range in mode mask 0x%x", bad);
            return MTTKRP_EINDEX;
        }
    }

    // Cold-row marks (common.cuh; unpacked records, N <= 3): degree of every index of every mode, and per mode the
    // degree below which a row is not among the K = MTTKRP_PREFETCH_ROWS most frequent ones (0 switches the marks off).
    for (int m = 0; m < N; ++m) { h->cold_deg[m] = 0; h->cold_rows[m] = 0; }
    const int64_t k_keep = h->knobs.prefetch_rows >= 0 ? h->knobs.prefetch_rows : 65536;
    const bool marks = nnz > 0 && N <= 3 && !h->packed && k_keep > 0;
    if (marks) {
        uint32_t hh[kDegBins];
        for (int m = 0; m < N; ++m) {
            const int64_t rows = h->dims[m];
            if (rows <= k_keep) continue;                        // every row is kept
            MK_CUDA(cudaMemsetAsync(degs[m], 0, 4 * (size_t)(rows + 1), st));
            MK_CUDA(cudaMemsetAsync(dhist, 0, 4 * kDegBins, st));
            k_count_keys_agg<<<grid_for(nnz, 256), 256, 0, st>>>((const uint32_t*)idx + (size_t)m * n, nnz, degs[m]);
            k_degree_hist<<<(unsigned)std::min<int64_t>(grid_for(rows, 256), 1024), 256, 0, st>>>(degs[m], rows, dhist);
            MK_CUDA(cudaMemcpyAsync(hh, dhist, 4 * kDegBins, cudaMemcpyDeviceToHost, st));
            MK_CUDA(cudaStreamSynchronize(st));
            // smallest bin boundary T with #{rows of degree >= T} <= K: rows of degree < T are cold
            int64_t cum = 0;
            int b = kDegBins;
            while (b > 0 && cum + hh[b - 1] <= k_keep) { cum += hh[b - 1]; --b; }
            h->cold_deg[m] = b >= kDegBins ? 0xffffffffu : deg_bin_floor(b);
            h->cold_rows[m] = rows - cum;
        }
    }

    for (int d = 0; d < N; ++d) {
        ModeMeta& mm = h->mode[d];
        uint32_t* dst = mm.next;   // holds perm_d until the maps are built
        if (nnz > 0) {
            uint32_t *ka = keyA, *kb = keyB, *pa = permA, *pb = permB;
            k_iota<<<grid_for(nnz, 256), 256, 0, st>>>(pa, nnz);
            for (int j = N - 1; j >= 0; --j) {
                const int m = mm.order[j];
                const uint32_t* col = (const uint32_t*)idx + (size_t)m * n;
                k_gather_u32<<<grid_for(nnz, 256), 256, 0, st>>>(col, pa, ka, nnz);
                const int bits = ceil_log2_i64(h->dims[m]);
                for (int shift = 0; shift < bits; shift += 8) {
                    k_radix_hist<<<(unsigned)nblocks, kSortThreads, 0, st>>>(ka, nnz, shift, hist, nblocks);
                    MK_TRY(exclusive_scan(hist, 256 * nblocks, sums, st));
                    k_radix_scatter<<<(unsigned)nblocks, kSortThreads, 0, st>>>(ka, pa, kb, pb, nnz, shift, hist, nblocks);
                    std::swap(ka, kb);
                    std::swap(pa, pb);
                }
                MK_CUDA(cudaGetLastError());
            }
            if (h->policy == 1) {
                // Alg. 1 policy: the partition of the output row becomes the leading sort key ("order the
                // hyperedges by partition id").  Degrees on the device, longest-first dealing on the host (as the paper
                // preprocesses on the CPU), then the radix passes over the partition id.
                const int64_t rows = h->dims[d];
                const uint32_t* col = (const uint32_t*)idx + (size_t)d * n;
                MK_CUDA(cudaMemsetAsync(flags, 0, 4 * (size_t)rows, st));
                k_count_keys<<<grid_for(nnz, 256), 256, 0, st>>>(col, nnz, flags);
                std::vector<int32_t> deg, part;
                std::vector<int64_t> loads;
                try { deg.resize((size_t)rows); part.resize((size_t)rows); loads.resize((size_t)h->kappa); }
                catch (...) { set_error("out of host memory"); return MTTKRP_EINVAL; }
                MK_CUDA(cudaMemcpyAsync(deg.data(), flags, 4 * (size_t)rows, cudaMemcpyDeviceToHost, st));
                MK_CUDA(cudaStreamSynchronize(st));
                if (!lpt_partition(deg.data(), rows, h->kappa, part.data(), loads.data())) { set_error("out of host memory"); return MTTKRP_EINVAL; }
                std::vector<uint32_t> bins((size_t)h->kappa + 1);
                bins[0] = 0;
                mm.max_bin = 0;
                mm.min_bin = nnz;
                for (int z = 0; z < h->kappa; ++z) {
                    bins[(size_t)z + 1] = bins[(size_t)z] + (uint32_t)loads[(size_t)z];
                    mm.max_bin = std::max(mm.max_bin, loads[(size_t)z]);
                    mm.min_bin = std::min(mm.min_bin, loads[(size_t)z]);
                }
                MK_CUDA(cudaMemcpyAsync(mm.bins, bins.data(), 4 * bins.size(), cudaMemcpyHostToDevice, st));
                MK_CUDA(cudaMemcpyAsync(flags2, part.data(), 4 * (size_t)rows, cudaMemcpyHostToDevice, st));
                k_gather_u32<<<grid_for(nnz, 256), 256, 0, st>>>(col, pa, ka, nnz);          // ka = i_d in the current order
                k_apply_table<<<grid_for(nnz, 256), 256, 0, st>>>(flags2, ka, nnz);          // ka = partition of that row
                const int pbits = ceil_log2_i64(h->kappa);
                for (int shift = 0; shift < pbits; shift += 8) {
                    k_radix_hist<<<(unsigned)nblocks, kSortThreads, 0, st>>>(ka, nnz, shift, hist, nblocks);
                    MK_TRY(exclusive_scan(hist, 256 * nblocks, sums, st));
                    k_radix_scatter<<<(unsigned)nblocks, kSortThreads, 0, st>>>(ka, pa, kb, pb, nnz, shift, hist, nblocks);
                    std::swap(ka, kb);
                    std::swap(pa, pb);
                }
                k_gather_u32<<<grid_for(nnz, 256), 256, 0, st>>>(col, pa, ka, nnz);          // ka = i_d in mode-d order again
                MK_CUDA(cudaStreamSynchronize(st));                                            // the host vectors go out of scope
                MK_CUDA(cudaGetLastError());
            }
            // pa = perm_d, ka = idx[d] in mode-d order
            {
                OrderArg oa;
                for (int l = 0; l < kMaxModes; ++l) oa.v[l] = mm.order[l];
                const int64_t nnz_pad = nshards * (int64_t)S;
                ColdArg ca;
                ca.deg[0] = ca.deg[1] = nullptr;
                ca.t[0] = ca.t[1] = 0;
                if (marks) {
                    const int ml = mm.order[N - 1];
                    if (h->cold_deg[ml]) { ca.deg[0] = degs[ml]; ca.t[0] = h->cold_deg[ml]; }
                    if (N == 3) { const int mf = mm.order[1]; if (h->cold_deg[mf]) { ca.deg[1] = degs[mf]; ca.t[1] = h->cold_deg[mf]; } }
                }
                k_build_flags<<<grid_for(nnz_pad, 256), 256, 0, st>>>(idx, pa, nnz, nnz_pad, N, oa, ca, mm.lflags);
            }
            MK_CUDA(cudaMemcpyAsync(dst, pa, 4 * n, cudaMemcpyDeviceToDevice, st));
            if (d == 0) MK_CUDA(cudaMemcpyAsync(h->perm0, pa, 4 * n, cudaMemcpyDeviceToDevice, st));

            // split rows (chains)
            if (nshards > 0) {
                k_chain_flags<<<grid_for(nshards + 1, 256), 256, 0, st>>>(ka, nnz, S, nshards, flags);
                MK_TRY(exclusive_scan(flags, nshards + 1, sums, st));
                k_chain_fill<<<grid_for(nshards, 256), 256, 0, st>>>(ka, nnz, S, nshards, flags, mm.chains);
                MK_CUDA(cudaMemcpyAsync(small + 8 + 2 * d, flags + nshards, 4, cudaMemcpyDeviceToDevice, st));
            }
            // empty rows
            const int64_t rows = h->dims[d];
            MK_CUDA(cudaMemsetAsync(flags, 0, 4 * (size_t)(rows + 1), st));
            k_mark_rows<<<grid_for(nnz, 256), 256, 0, st>>>(ka, nnz, flags);
            k_invert_flags<<<grid_for(rows + 1, 256), 256, 0, st>>>(flags, rows);
            MK_TRY(exclusive_scan(flags, rows + 1, sums, st));
            k_compact_ids<<<grid_for(rows, 256), 256, 0, st>>>(flags, rows, mm.empty_rows);
            MK_CUDA(cudaMemcpyAsync(small + 8 + 2 * d + 1, flags + rows, 4, cudaMemcpyDeviceToDevice, st));
            MK_CUDA(cudaGetLastError());
        } else {
            // no nonzeros: every row is empty
            const int64_t rows = h->dims[d];
            k_iota<<<grid_for(rows, 256), 256, 0, st>>>(mm.empty_rows, rows);
            MK_CUDA(cudaGetLastError());
        }
    }

    if (nnz > 0) {
        // tensor copy in mode-0 order
        OrderArg oa;
        for (int l = 0; l < kMaxModes; ++l) oa.v[l] = h->mode[0].order[l];
        const int64_t nnz_pad = nshards * (int64_t)S;
        if (h->packed) {
            uint4* rec = reinterpret_cast<uint4*>(h->rec_cur);
            const unsigned g = grid_for(nnz_pad, 256);
            const PackDesc pd = h->mode[0].pk;
            switch (N) {
                case 4: k_build_records_pk<4><<<g, 256, 0, st>>>(idx, vals, h->perm0, h->mode[0].lflags, nnz, nnz_pad, oa, pd, rec); break;
                case 5: k_build_records_pk<5><<<g, 256, 0, st>>>(idx, vals, h->perm0, h->mode[0].lflags, nnz, nnz_pad, oa, pd, rec); break;
                case 6: k_build_records_pk<6><<<g, 256, 0, st>>>(idx, vals, h->perm0, h->mode[0].lflags, nnz, nnz_pad, oa, pd, rec); break;
                case 7: k_build_records_pk<7><<<g, 256, 0, st>>>(idx, vals, h->perm0, h->mode[0].lflags, nnz, nnz_pad, oa, pd, rec); break;
                case 8: k_build_records_pk<8><<<g, 256, 0, st>>>(idx, vals, h->perm0, h->mode[0].lflags, nnz, nnz_pad, oa, pd, rec); break;
                default: set_error("packed records need nmodes >= 4"); return MTTKRP_EINVAL;
            }
        } else {
            k_build_records<<<grid_for(nnz_pad, 256), 256, 0, st>>>(idx, vals, h->perm0, h->mode[0].lflags, nnz, nnz_pad, N, oa, h->rec_cur);
        }
        // Slot d still holds perm_d; go d = 0..N-1, the last one needs perm_0, which slot 0 no longer
        // holds -> use the perm0 copy.
        uint32_t* inv = keyA;
        for (int d = 0; d < N; ++d) {
            const int e = (d + 1) % N;
            const uint32_t* perm_e = (e == 0) ? h->perm0 : h->mode[e].next;
            // gather map: slot d <- inv_d[perm_e[j]] = position in layout d of element j of layout e
            k_invert<<<grid_for(nnz, 256), 256, 0, st>>>(h->mode[d].next, inv, nnz);
            k_gather_u32<<<grid_for(nnz, 256), 256, 0, st>>>(inv, perm_e, h->mode[d].next, nnz);
        }
        if (h->fuse) {
            // Scatter form of every transition for the fused kernel (Alg. 3 as written): scat_d = next_d^-1
            // is the remap id of mode (d+1)%N, sflags_d the next layout's run-end flags read through it.
            for (int d = 0; d < N; ++d) {
                k_invert<<<grid_for(nnz, 256), 256, 0, st>>>(h->mode[d].next, h->mode[d].scat, nnz);
                k_gather_u8<<<grid_for(nnz, 256), 256, 0, st>>>(h->mode[(d + 1) % N].lflags, h->mode[d].scat, h->mode[d].sflags, nnz);
            }
        }
        MK_CUDA(cudaGetLastError());
        // Blocked remap order (remap.cu): destination positions of the remap d -> d+1 grouped, stably,
        // by the source block they read from: one 8-bit radix pass on the block id.  The block is sized
        // to stay L2-resident while the whole grid gathers from it.
        int block_log2 = h->knobs.remap_block_log2 >= 0 ? h->knobs.remap_block_log2 : 20;   // knob clamped to [10,26]
        while ((nnz >> block_log2) > 255) ++block_log2;                // at most 256 blocks (one radix digit)
        for (int d = 0; d < N; ++d) {
            ModeMeta& mm = h->mode[d];
            mm.block_log2 = block_log2;
            k_block_keys<<<grid_for(nnz, 256), 256, 0, st>>>(mm.next, block_log2, keyA, nnz);
            k_iota<<<grid_for(nnz, 256), 256, 0, st>>>(permA, nnz);
            k_radix_hist<<<(unsigned)nblocks, kSortThreads, 0, st>>>(keyA, nnz, 0, hist, nblocks);
            MK_TRY(exclusive_scan(hist, 256 * nblocks, sums, st));
            k_radix_scatter<<<(unsigned)nblocks, kSortThreads, 0, st>>>(keyA, permA, keyB, mm.ord, nnz, 0, hist, nblocks);
            k_gather_u32<<<grid_for(nnz, 256), 256, 0, st>>>(mm.next, mm.ord, mm.osrc, nnz);
            k_count_breaks<<<grid_for(nnz, 256), 256, 0, st>>>(mm.ord, nnz, small + 32 + d);
            k_count_breaks<<<grid_for(nnz, 256), 256, 0, st>>>(mm.next, nnz, small + 40 + d);
        }
        MK_CUDA(cudaGetLastError());
    }

    uint32_t counts[2 * kMaxModes] = {0}, breaks[2 * kMaxModes] = {0};
    MK_CUDA(cudaMemcpyAsync(counts, small + 8, sizeof(uint32_t) * 2 * N, cudaMemcpyDeviceToHost, st));
    MK_CUDA(cudaMemcpyAsync(breaks, small + 32, sizeof(uint32_t) * 2 * kMaxModes, cudaMemcpyDeviceToHost, st));
    MK_CUDA(cudaStreamSynchronize(st));
    const int benv = h->knobs.remap_blocked;                     // 0 / 1 force the choice (experiments), -1: decide here
    for (int d = 0; d < N; ++d) {
        h->mode[d].n_chains = (nnz > 0 && h->policy == 0) ? counts[2 * d] : 0;   // Alg. 1 policy: no row spans blocks
        h->mode[d].n_empty = nnz > 0 ? counts[2 * d + 1] : h->dims[d];
        // Use the blocked order when the source window fits L2 comfortably, the destination runs are
        // long enough to store whole sectors (average run >= 4 records), and the plain walk is a random
        // gather (when consecutive destinations read consecutive sources - a remap that moves whole
        // fibers - the plain walk is already sequential on both sides).
        const int64_t runs = (int64_t)breaks[d] + 1;
        const int64_t src_runs = (int64_t)breaks[kMaxModes + d] + 1;
        const bool fits = ((int64_t)h->rec_words * 4 << h->mode[d].block_log2) <= (48ll << 20);
        bool blocked = nnz > 0 && fits && (nnz >> h->mode[d].block_log2) >= 2 && nnz / runs >= 4 &&
                       (double)nnz / (double)src_runs < 1.5;
        if (benv >= 0) blocked = nnz > 0 && benv == 1;
        h->mode[d].blocked = blocked ? 1 : 0;
        h->mode[d].avg_run = nnz > 0 ? (double)nnz / (double)runs : 0.0;
        h->mode[d].plain_ms = h->mode[d].twopass_ms = 0.f;
    }
    // Two-pass remap for the transitions that stay a random gather (16-byte records, tensors of many windows): build
    // the two maps into the (otherwise unused) ord / osrc arrays, then TIME cycles of transitions with the plain
    // walk and with the two passes on the real tensor and keep, per transition, the faster one (medians, below).
    const int tenv = h->knobs.remap_twopass;                    // 0 / 1 force the choice (tests, experiments)
    const bool tp_forced_on = tenv == 1, tp_forced_off = tenv == 0 || benv >= 0;
    bool cand[kMaxModes] = {false};
    bool any_cand = false;
    if (nnz > 0 && h->rec_words == 4 && !tp_forced_off) {
        int wlog = h->knobs.twopass_window_log2 >= 0 ? h->knobs.twopass_window_log2 : kTwoPassWindowLog2;   // knob: tests
        while ((nnz >> wlog) > 255) ++wlog;
        for (int d = 0; d < N; ++d) {
            const int64_t src_runs = (int64_t)breaks[kMaxModes + d] + 1;
            const bool random_gather = (double)nnz / (double)src_runs < 1.5;
            cand[d] = !h->mode[d].blocked && (tp_forced_on || (random_gather && (nnz >> wlog) >= 8));
            if (!cand[d]) continue;
            any_cand = true;
            ModeMeta& mm = h->mode[d];
            mm.block_log2 = wlog;                                     // two-pass walk: log2 of the destination window
            uint32_t* scat = permB;                                   // inverse of next: destination of source position s
            k_invert<<<grid_for(nnz, 256), 256, 0, st>>>(mm.next, scat, nnz);
            k_block_keys<<<grid_for(nnz, 256), 256, 0, st>>>(scat, wlog, keyA, nnz);
            k_iota<<<grid_for(nnz, 256), 256, 0, st>>>(permA, nnz);
            k_radix_hist<<<(unsigned)nblocks, kSortThreads, 0, st>>>(keyA, nnz, 0, hist, nblocks);
            MK_TRY(exclusive_scan(hist, 256 * nblocks, sums, st));
            // mm.osrc = source positions grouped (stably) by destination window = the order of the intermediate copy
            k_radix_scatter<<<(unsigned)nblocks, kSortThreads, 0, st>>>(keyA, permA, keyB, mm.osrc, nnz, 0, hist, nblocks);
            k_invert<<<grid_for(nnz, 256), 256, 0, st>>>(mm.osrc, mm.ord, nnz);                    // s1[s] = slot of source s
            k_invert_through<<<grid_for(nnz, 256), 256, 0, st>>>(mm.osrc, scat, keyA, nnz);        // g2[t] = slot of destination t
            MK_CUDA(cudaMemcpyAsync(mm.osrc, keyA, 4 * n, cudaMemcpyDeviceToDevice, st));
        }
        MK_CUDA(cudaGetLastError());
    }
    if (any_cand) {
        // One warm-up cycle, then kReps plain cycles and kReps two-pass cycles, alternating; per transition the MEDIAN
        // of each walk decides (one sample per walk let a single disturbed run flip the choice).  The events are
        // destroyed on every exit path; a failing create deletes the handle, so `blocked` needs no restoring there.
        struct EventPair {
            cudaEvent_t a = nullptr, b = nullptr;
            ~EventPair() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); }
        } ev;
        MK_CUDA(cudaEventCreate(&ev.a));
        MK_CUDA(cudaEventCreate(&ev.b));
        constexpr int kReps = 3;
        int keep[kMaxModes];
        float t_plain[kMaxModes][kReps], t_two[kMaxModes][kReps];
        for (int d = 0; d < N; ++d) keep[d] = h->mode[d].blocked == 1 ? 1 : 0;
        for (int cyc = 0; cyc < 1 + 2 * kReps; ++cyc) {
            const bool two = cyc > 0 && cyc % 2 == 0;           // cycles 1, 3, 5 plain; 2, 4, 6 two passes
            for (int d = 0; d < N; ++d) {
                h->mode[d].blocked = (two && cand[d]) ? 2 : keep[d];
                MK_CUDA(cudaEventRecord(ev.a, st));
                MK_TRY(launch_remap(h, d, (d + 1) % N, nullptr, st));
                MK_CUDA(cudaEventRecord(ev.b, st));
                MK_CUDA(cudaEventSynchronize(ev.b));
                float ms = 0.f;
                MK_CUDA(cudaEventElapsedTime(&ms, ev.a, ev.b));
                if (cyc > 0) (two ? t_two : t_plain)[d][(cyc - 1) / 2] = ms;
            }
        }
        auto median3 = [](const float* t) { return std::max(std::min(t[0], t[1]), std::min(std::max(t[0], t[1]), t[2])); };
        for (int d = 0; d < N; ++d) {
            h->mode[d].blocked = keep[d];
            if (!cand[d]) continue;
            h->mode[d].plain_ms = median3(t_plain[d]);
            h->mode[d].twopass_ms = median3(t_two[d]);
            h->mode[d].blocked = (tp_forced_on || h->mode[d].twopass_ms < 0.95f * h->mode[d].plain_ms) ? 2 : 0;
        }
        h->remaps_done = 0;                                      // the tensor is back in the mode-0 layout (N transitions per cycle)
    }
    // Give back what the chosen walks do not need: the slot pairs of the transitions that read ord / osrc move to the
    // front of the pool (lower addresses only, in mode order, on the stream: a destination slot was vacated or never
    // used), the other modes lose their pointers, and the handle holds the workspace up to the last used slot.
    int used = 0;
    for (int d = 0; d < N; ++d) {
        ModeMeta& mm = h->mode[d];
        if (nnz > 0 && mm.blocked != 0) {
            uint32_t* o = reinterpret_cast<uint32_t*>(ws + plan.pool + (size_t)(2 * used) * plan.pool_slot);
            uint32_t* s2 = reinterpret_cast<uint32_t*>(ws + plan.pool + (size_t)(2 * used + 1) * plan.pool_slot);
            if (o != mm.ord) {
                MK_CUDA(cudaMemcpyAsync(o, mm.ord, 4 * n, cudaMemcpyDeviceToDevice, st));
                MK_CUDA(cudaMemcpyAsync(s2, mm.osrc, 4 * n, cudaMemcpyDeviceToDevice, st));
            }
            mm.ord = o;
            mm.osrc = s2;
            ++used;
        } else {
            mm.ord = mm.osrc = nullptr;
        }
    }
    const size_t rec_bytes = (size_t)h->rec_words * 4 * (size_t)(nshards * S);
    h->bytes_held = (int64_t)(used ? plan.pool + (size_t)(2 * used) * plan.pool_slot : plan.persistent_end + rec_bytes);
    return MTTKRP_OK;
}

}  // namespace mk
