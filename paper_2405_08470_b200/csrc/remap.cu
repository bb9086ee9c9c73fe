// Dynamic tensor remapping (Alg. 3).  The paper scatters, T_out[b_out] = x_i with
// b_out the element's remap id for mode (d+1) mod N; every element has a unique
// destination (Observation 1).  Here the same permutation is applied in gather
// form, T_out[j] = T_in[prev[j]]: stores are coalesced and whole 32-byte sectors, the random side is
// the 16-byte loads.  On B200 the scatter form measured 2.3x slower (partial-sector writes turn
// into read-modify-write in DRAM; kernel v1 of round 1).
// Records are role-ordered (sort keys major to minor, then the value), so the pass also permutes
// the index fields from the source layout's key order to the destination's, refreshes the
// zero-valued padding records that fill the last shard, and merges the destination layout's
// precomputed run-end flags into bit 31 of the key words (common.cuh), which saves the MTTKRP
// kernel every look-ahead compare.
#include "common.cuh"

namespace mk {


// 3-mode records are 16 B: one 128-bit load and one 128-bit store per nonzero.
// BLOCKED: thread t handles destination position ord[t] instead of t.  `ord` lists the destination
// positions grouped by the source block (2^block_log2 records) their record comes from, so at any
// time the whole grid gathers from one source window that stays in L2, and every 64-byte DRAM
// fetch is used completely; inside a group the destination positions ascend in long runs (the
// layouts' key orders are chosen for that, build.cu choose_key_order), so the stores stay whole sectors.
// Independent gather chains in flight per thread: 4 for the blocked walk (L2 hits), 8 for the plain walk (random
// HBM reads need more parallelism); measured on configs[1] / configs[2].
template <bool BLOCKED>
__host__ __device__ constexpr int remap_per_thread() { return BLOCKED ? 4 : 8; }

template <bool BLOCKED>
__global__ void __launch_bounds__(256) k_remap3(const uint4* __restrict__ in, const uint32_t* __restrict__ prev,
                                                const uint32_t* __restrict__ ord, const uint32_t* __restrict__ osrc,
                                                const uint8_t* __restrict__ dflags, uint4* __restrict__ out, int64_t nnz,
                                                int64_t nnz_pad, FieldMap fm, int64_t t0) {
    constexpr int U = remap_per_thread<BLOCKED>();
    const int64_t base = t0 + (int64_t)blockIdx.x * (256 * U) + threadIdx.x;     // t0 > 0: only the tail (padding) positions
    int64_t j[U];
    uint32_t src[U], fl[U];
    uint4 r[U];
#pragma unroll
    for (int i = 0; i < U; ++i) {
        const int64_t t = base + i * 256;
        j[i] = (BLOCKED && t < nnz) ? (int64_t)__ldcs(ord + t) : t;          // padding positions are handled in place
        if (t >= nnz_pad) j[i] = -1;
        if (BLOCKED && t < nnz) src[i] = __ldcs(osrc + t);
        else src[i] = __ldcs(prev + (t < nnz ? t : nnz - 1));
    }
#pragma unroll
    for (int i = 0; i < U; ++i) fl[i] = j[i] < 0 ? 0u : dflags[j[i]];
#pragma unroll
    for (int i = 0; i < U; ++i) r[i] = __ldg(in + src[i]);
#pragma unroll
    for (int i = 0; i < U; ++i) {
        if (j[i] < 0) continue;
        const uint32_t f[3] = {r[i].x & kKeyMask, r[i].y & kKeyMask, r[i].z & kKeyMask};
        uint32_t k[3];
#pragma unroll
        for (int l = 0; l < 3; ++l) k[l] = fm.src[l] == 0 ? f[0] : (fm.src[l] == 1 ? f[1] : f[2]);
        apply_run_flags<3>(k, fl[i]);
        __stcs(out + j[i], make_uint4(k[0], k[1], k[2], j[i] < nnz ? r[i].w : 0u));
    }
}

template <int N, bool BLOCKED>
__global__ void __launch_bounds__(256) k_remap(const uint32_t* __restrict__ in, const uint32_t* __restrict__ prev,
                                               const uint32_t* __restrict__ ord, const uint8_t* __restrict__ dflags,
                                               uint32_t* __restrict__ out, int64_t nnz, int64_t nnz_pad, FieldMap fm) {
    constexpr int U = remap_per_thread<BLOCKED>();
    const int64_t base = (int64_t)blockIdx.x * (256 * U) + threadIdx.x;
    int64_t j[U];
    const uint32_t* r[U];
#pragma unroll
    for (int i = 0; i < U; ++i) {
        const int64_t t = base + i * 256;
        j[i] = (BLOCKED && t < nnz) ? (int64_t)__ldcs(ord + t) : t;
        if (t >= nnz_pad) j[i] = -1;
    }
#pragma unroll
    for (int i = 0; i < U; ++i) {
        const int64_t jj = j[i] < 0 ? 0 : (j[i] < nnz ? j[i] : nnz - 1);
        r[i] = in + (size_t)__ldg(prev + jj) * (N + 1);
    }
#pragma unroll
    for (int i = 0; i < U; ++i) {
        if (j[i] < 0) continue;
        uint32_t k[N];
#pragma unroll
        for (int l = 0; l < N; ++l) k[l] = __ldg(r[i] + fm.src[l]) & kKeyMask;
        const uint32_t val = j[i] < nnz ? __ldg(r[i] + N) : 0u;
        apply_run_flags<N>(k, dflags[j[i]]);
        uint32_t* o = out + (size_t)j[i] * (N + 1);
#pragma unroll
        for (int l = 0; l < N; ++l) o[l] = k[l];
        o[N] = val;
    }
}

// Packed 16-byte records (common.cuh PackDesc), any N >= 4: one 128-bit load and store per nonzero.  The host
// composes, per destination level, where its key sits in the SOURCE record (RemapPk), so the kernel unpacks
// straight into destination order and repacks with the destination layout's offsets and flags.

template <int N, bool BLOCKED>
__global__ void __launch_bounds__(256) k_remap_pk(const uint4* __restrict__ in, const uint32_t* __restrict__ prev,
                                                  const uint32_t* __restrict__ ord, const uint32_t* __restrict__ osrc,
                                                  const uint8_t* __restrict__ dflags, uint4* __restrict__ out, int64_t nnz,
                                                  int64_t nnz_pad, RemapPk rp, PackDesc dd, int64_t t0) {
    constexpr int U = remap_per_thread<BLOCKED>();
    const int64_t base = t0 + (int64_t)blockIdx.x * (256 * U) + threadIdx.x;
    int64_t j[U];
    uint32_t src[U], fl[U];
    uint4 r[U];
#pragma unroll
    for (int i = 0; i < U; ++i) {
        const int64_t t = base + i * 256;
        j[i] = (BLOCKED && t < nnz) ? (int64_t)__ldcs(ord + t) : t;
        if (t >= nnz_pad) j[i] = -1;
        if (BLOCKED && t < nnz) src[i] = __ldcs(osrc + t);
        else src[i] = __ldcs(prev + (t < nnz ? t : nnz - 1));
    }
#pragma unroll
    for (int i = 0; i < U; ++i) fl[i] = j[i] < 0 ? 0u : dflags[j[i]];
#pragma unroll
    for (int i = 0; i < U; ++i) r[i] = __ldg(in + src[i]);
#pragma unroll
    for (int i = 0; i < U; ++i) {
        if (j[i] < 0) continue;
        uint32_t k[N];
#pragma unroll
        for (int l = 0; l < N; ++l)
            k[l] = rp.soff[l] < 0 ? (r[i].z & rp.smask[l]) : pk_get(r[i].x, r[i].y, rp.soff[l], rp.smask[l]);
        __stcs(out + j[i], pk_pack<N>(k, fl[i], j[i] < nnz ? r[i].w : 0u, dd));
    }
}

// The walk of one remap pass: `map[j]` = source position of destination position j; blocked walks also carry
// `ord` / `osrc` (see k_remap3).
struct Walk { const uint32_t* map; const uint32_t* ord; const uint32_t* osrc; int blocked; };

template <int N>
static void launch_remap_n(mttkrp_handle_s* h, int from, int to, const Walk& w, unsigned grid, int64_t nnz_pad, const FieldMap& fm, cudaStream_t st,
                           int64_t t0 = 0) {
    const ModeMeta& mf = h->mode[from];
    const uint8_t* dflags = h->mode[to].lflags;
    if constexpr (N == 3) {
        if (w.blocked) k_remap3<true><<<grid, 256, 0, st>>>((const uint4*)h->rec_cur, w.map, w.ord, w.osrc, dflags, (uint4*)h->rec_alt, h->nnz, nnz_pad, fm, t0);
        else k_remap3<false><<<grid, 256, 0, st>>>((const uint4*)h->rec_cur, w.map, w.ord, w.osrc, dflags, (uint4*)h->rec_alt, h->nnz, nnz_pad, fm, t0);
    } else {
        if constexpr (N >= 4) {
            if (h->packed) {
                FieldMap fm2;
                RemapPk rp;
                remap_fields(h, from, to, &fm2, &rp);
                const PackDesc dd = h->mode[to].pk;
                if (w.blocked) k_remap_pk<N, true><<<grid, 256, 0, st>>>((const uint4*)h->rec_cur, w.map, w.ord, w.osrc, dflags, (uint4*)h->rec_alt, h->nnz, nnz_pad, rp, dd, t0);
                else k_remap_pk<N, false><<<grid, 256, 0, st>>>((const uint4*)h->rec_cur, w.map, w.ord, w.osrc, dflags, (uint4*)h->rec_alt, h->nnz, nnz_pad, rp, dd, t0);
                return;
            }
        }
        if (w.blocked) k_remap<N, true><<<grid, 256, 0, st>>>(h->rec_cur, w.map, w.ord, dflags, h->rec_alt, h->nnz, nnz_pad, fm);
        else k_remap<N, false><<<grid, 256, 0, st>>>(h->rec_cur, w.map, w.ord, dflags, h->rec_alt, h->nnz, nnz_pad, fm);
    }
}

// Pass 1 of the two-pass remap (16-byte records): mid[s1[s]] = in[s].  The intermediate copy groups the records by
// the 2^21-record window of the destination layout they go to, in source order inside a window: the source is read
// once, sequentially, and every block appends a contiguous run to each of the ~100 window streams, which L2 merges
// into whole lines.  Pass 2 is the plain gather walk out of `mid`: its random reads stay inside one window (32 MB).
// A block takes a tile of kScatterTile consecutive source records.  Inside a window the intermediate order is the
// source order, so the tile's records for one window occupy CONSECUTIVE slots of `mid`: the block sorts its tile by
// window in shared memory (histogram + first slot per window) and then writes it out in that order, consecutive lanes
// to consecutive addresses, i.e. whole sectors and lines instead of 16-byte pieces.
constexpr int kScatterTile = 2048;
__global__ void __launch_bounds__(256) k_scatter16(const uint4* __restrict__ in, const uint32_t* __restrict__ s1,
                                                   uint4* __restrict__ mid, int64_t nnz, int wlog) {
    __shared__ uint4 s_rec[kScatterTile];
    __shared__ uint32_t s_dst[kScatterTile];
    __shared__ uint32_t s_cnt[256], s_first[256], s_off[256];
    const int64_t base = (int64_t)blockIdx.x * kScatterTile;
    const int n = (int)min((int64_t)kScatterTile, nnz - base);
    s_cnt[threadIdx.x] = 0;
    s_first[threadIdx.x] = 0xffffffffu;
    __syncthreads();
    constexpr int PER = kScatterTile / 256;
    uint4 r[PER];
    uint32_t dst[PER];
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const int j = threadIdx.x + i * 256;
        if (j < n) {
            dst[i] = __ldcs(s1 + base + j);
            r[i] = __ldcs(in + base + j);
            const uint32_t w = dst[i] >> wlog;
            atomicAdd(&s_cnt[w], 1u);
            atomicMin(&s_first[w], dst[i]);
        }
    }
    __syncthreads();
    {   // exclusive scan of the 256 window counts (one warp, 8 per lane)
        if (threadIdx.x < 32) {
            uint32_t v[8], sum = 0;
#pragma unroll
            for (int q = 0; q < 8; ++q) { v[q] = s_cnt[threadIdx.x * 8 + q]; sum += v[q]; }
            uint32_t inc = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
                if ((int)threadIdx.x >= o) inc += t;
            }
            uint32_t run = inc - sum;
#pragma unroll
            for (int q = 0; q < 8; ++q) { s_off[threadIdx.x * 8 + q] = run; run += v[q]; }
        }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const int j = threadIdx.x + i * 256;
        if (j < n) {
            const uint32_t w = dst[i] >> wlog;
            const uint32_t slot = s_off[w] + (dst[i] - s_first[w]);
            s_rec[slot] = r[i];
            s_dst[slot] = dst[i];
        }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < n; j += 256) mid[s_dst[j]] = s_rec[j];
}

void remap_fields(const mttkrp_handle_s* h, int from, int to, FieldMap* fm, RemapPk* rp) {
    const int N = h->N;
    const ModeMeta& mf = h->mode[from];
    for (int l = 0; l < kMaxModes; ++l) { fm->src[l] = 0; rp->soff[l] = 0; rp->smask[l] = 0; }
    for (int l = 0; l < N; ++l) {
        const int sl = mf.pos[h->mode[to].order[l]];
        fm->src[l] = sl;
        if (h->packed) {
            rp->soff[l] = (sl == N - 1) ? -1 : mf.pk.off[sl];
            rp->smask[l] = pk_mask(mf.pk.bits[sl]);
        }
    }
}

// One gather pass from layout `from` into layout `to`, then swap(T_in, T_out).  jump == nullptr: the stored
// walk of the transition from -> (from+1)%N (the paper's only case).  Otherwise `jump[j]` is the
// position in layout `from` of the element at position j of layout `to` (composed by api.cu for out-of-order
// calls): plain walk in destination order.
mttkrp_status_t launch_remap(mttkrp_handle_s* h, int from, int to, const uint32_t* jump, cudaStream_t st) {
    const int N = h->N;
    if (h->nnz > 0) {
        const ModeMeta& mf = h->mode[from];
        Walk w;
        if (jump) { w.map = jump; w.ord = nullptr; w.osrc = nullptr; w.blocked = 0; }
        else if (mf.blocked == 2) {
            // two passes: group by destination window into the other copy, then gather out of it into this one
            TimedLaunch tl(h->timing, kClsRemap, st);
            k_scatter16<<<(unsigned)((h->nnz + kScatterTile - 1) / kScatterTile), 256, 0, st>>>((const uint4*)h->rec_cur, mf.ord, (uint4*)h->rec_alt, h->nnz,
                                                                                           mf.block_log2);
            uint32_t* t = h->rec_cur; h->rec_cur = h->rec_alt; h->rec_alt = t;
            w.map = mf.osrc; w.ord = nullptr; w.osrc = nullptr; w.blocked = 0;
        }
        else { w.map = mf.next; w.ord = mf.ord; w.osrc = mf.osrc; w.blocked = mf.blocked; }
        FieldMap fm;
        RemapPk rp_unused;
        remap_fields(h, from, to, &fm, &rp_unused);
        const int64_t nnz_pad = h->num_shards * (int64_t)h->shard_nnz;
        const int per_block = 256 * (w.blocked ? remap_per_thread<true>() : remap_per_thread<false>());
        const unsigned grid = (unsigned)((nnz_pad + per_block - 1) / per_block);
        TimedLaunch tl(h->timing, kClsRemap, st);
        switch (N) {
            case 2: launch_remap_n<2>(h, from, to, w, grid, nnz_pad, fm, st); break;
            case 3: launch_remap_n<3>(h, from, to, w, grid, nnz_pad, fm, st); break;
            case 4: launch_remap_n<4>(h, from, to, w, grid, nnz_pad, fm, st); break;
            case 5: launch_remap_n<5>(h, from, to, w, grid, nnz_pad, fm, st); break;
            case 6: launch_remap_n<6>(h, from, to, w, grid, nnz_pad, fm, st); break;
            case 7: launch_remap_n<7>(h, from, to, w, grid, nnz_pad, fm, st); break;
            case 8: launch_remap_n<8>(h, from, to, w, grid, nnz_pad, fm, st); break;
            default: set_error("remap: unsupported nmodes %d", N); return MTTKRP_EUNSUPPORTED;
        }
        MK_CUDA(cudaGetLastError());
    }
    uint32_t* t = h->rec_cur;      // swap(T_in, T_out), Alg. 5 line 12
    h->rec_cur = h->rec_alt;
    h->rec_alt = t;
    h->cur = to;
    h->remaps_done++;
    return MTTKRP_OK;
}

// MTTKRP_FUSE: the MTTKRP kernel scattered the nnz real records of layout `to` into rec_alt; this writes the
// zero-valued padding records that fill the last shard (16-byte records only, plain walk from position nnz on).
mttkrp_status_t launch_remap_padding(mttkrp_handle_s* h, int from, int to, cudaStream_t st) {
    const int64_t nnz_pad = h->num_shards * (int64_t)h->shard_nnz;
    if (h->nnz == 0 || nnz_pad == h->nnz) return MTTKRP_OK;
    const ModeMeta& mf = h->mode[from];
    Walk w;
    w.map = mf.next; w.ord = nullptr; w.osrc = nullptr; w.blocked = 0;
    FieldMap fm;
    RemapPk rp_unused;
    remap_fields(h, from, to, &fm, &rp_unused);
    const int per_block = 256 * remap_per_thread<false>();
    const unsigned grid = (unsigned)((nnz_pad - h->nnz + per_block - 1) / per_block);
    switch (h->N) {
        case 3: launch_remap_n<3>(h, from, to, w, grid, nnz_pad, fm, st, h->nnz); break;
        case 4: launch_remap_n<4>(h, from, to, w, grid, nnz_pad, fm, st, h->nnz); break;
        case 5: launch_remap_n<5>(h, from, to, w, grid, nnz_pad, fm, st, h->nnz); break;
        case 6: launch_remap_n<6>(h, from, to, w, grid, nnz_pad, fm, st, h->nnz); break;
        case 7: launch_remap_n<7>(h, from, to, w, grid, nnz_pad, fm, st, h->nnz); break;
        case 8: launch_remap_n<8>(h, from, to, w, grid, nnz_pad, fm, st, h->nnz); break;
        default: set_error("fused remap: unsupported nmodes %d", h->N); return MTTKRP_EUNSUPPORTED;
    }
    MK_CUDA(cudaGetLastError());
    return MTTKRP_OK;
}

// Carries the original-position array from one layout to the next: out[j] = in[prev[j]].
__global__ void k_perm_step(const uint32_t* __restrict__ prev, const uint32_t* __restrict__ in,
                            uint32_t* __restrict__ out, int64_t nnz) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < nnz) out[j] = in[prev[j]];
}

mttkrp_status_t launch_perm_step(const uint32_t* prev, const uint32_t* in, uint32_t* out, int64_t nnz, cudaStream_t st) {
    if (nnz > 0) {
        k_perm_step<<<(unsigned)((nnz + 255) / 256), 256, 0, st>>>(prev, in, out, nnz);
        MK_CUDA(cudaGetLastError());
    }
    return MTTKRP_OK;
}

struct PosArg { int v[kMaxModes]; };

__global__ void k_export(const uint32_t* __restrict__ rec, int64_t nnz, int N, PosArg pos, int32_t* __restrict__ idx,
                         float* __restrict__ vals) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nnz) return;
    const uint32_t* r = rec + (size_t)k * (N + 1);
    for (int m = 0; m < N; ++m) idx[(size_t)m * nnz + k] = (int32_t)(r[pos.v[m]] & kKeyMask);
    vals[k] = __uint_as_float(r[N]);
}

// packed records: pos.v[m] = level of mode m in the resident layout
__global__ void k_export_pk(const uint4* __restrict__ rec, int64_t nnz, int N, PosArg pos, PackDesc pd,
                            int32_t* __restrict__ idx, float* __restrict__ vals) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nnz) return;
    const uint4 r = rec[k];
    for (int m = 0; m < N; ++m) {
        const int l = pos.v[m];
        const uint32_t mask = pk_mask(pd.bits[l]);
        idx[(size_t)m * nnz + k] = (int32_t)(l == N - 1 ? (r.z & mask) : pk_get(r.x, r.y, pd.off[l], mask));
    }
    vals[k] = __uint_as_float(r.w);
}

mttkrp_status_t launch_export(const mttkrp_handle_s* h, int32_t* idx, float* vals, cudaStream_t st) {
    if (h->nnz > 0) {
        PosArg pa;
        for (int m = 0; m < kMaxModes; ++m) pa.v[m] = h->mode[h->cur].pos[m];
        const unsigned grid = (unsigned)((h->nnz + 255) / 256);
        if (h->packed) k_export_pk<<<grid, 256, 0, st>>>((const uint4*)h->rec_cur, h->nnz, h->N, pa, h->mode[h->cur].pk, idx, vals);
        else k_export<<<grid, 256, 0, st>>>(h->rec_cur, h->nnz, h->N, pa, idx, vals);
        MK_CUDA(cudaGetLastError());
    }
    return MTTKRP_OK;
}

// Row degrees of one mode from the resident copy (Alg. 1's vertex degrees): level = position of
// that mode in the resident layout's key order.  Off the hot path; global atomics are fine here.
__global__ void k_row_degrees(const uint32_t* __restrict__ rec, int64_t nnz, int rec_words, int packed, int N, int level,
                              PackDesc pd, int32_t* __restrict__ deg) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nnz) return;
    const uint32_t* r = rec + (size_t)k * rec_words;
    uint32_t key;
    if (packed) key = level == N - 1 ? (r[2] & pk_mask(pd.bits[level])) : pk_get(r[0], r[1], pd.off[level], pk_mask(pd.bits[level]));
    else key = r[level] & kKeyMask;
    atomicAdd(deg + key, 1);
}

mttkrp_status_t launch_row_degrees(const mttkrp_handle_s* h, int d, int32_t* deg_dev, cudaStream_t st) {
    MK_CUDA(cudaMemsetAsync(deg_dev, 0, sizeof(int32_t) * (size_t)h->dims[d], st));
    if (h->nnz > 0) {
        const ModeMeta& mm = h->mode[h->cur];
        k_row_degrees<<<(unsigned)((h->nnz + 255) / 256), 256, 0, st>>>(h->rec_cur, h->nnz, h->rec_words, h->packed, h->N,
                                                                         mm.pos[d], mm.pk, deg_dev);
        MK_CUDA(cudaGetLastError());
    }
    return MTTKRP_OK;
}

}  // namespace mk
