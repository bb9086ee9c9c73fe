// Dynamic tensor remapping (Alg. 3).  The paper scatters, T_out[b_out] = x_i with
// b_out the element's remap id for mode (d+1) mod N; every element has a unique
// destination (Observation 1).  Here the same permutation is applied in gather
// form, T_out[j] = T_in[prev[j]]: stores are coalesced and whole 32-byte sectors, the random side is
// the 16-byte loads.  On B200 the scatter form measured 2.3x slower (partial-sector writes turn
// into read-modify-write in DRAM; profiles/r1_v1_ncu_summary.md).
// Records are role-ordered (sort keys major to minor, then the value), so the pass also permutes
// the index fields from the source layout's key order to the destination's, refreshes the
// zero-valued padding records that fill the last shard, and merges the destination layout's
// precomputed run-end flags into bit 31 of the key words (common.cuh), which saves the MTTKRP
// kernel every look-ahead compare.
#include "common.cuh"

namespace mk {

struct FieldMap { int src[kMaxModes]; };   // out.field[l] = in.field[src[l]]

// 3-mode records are 16 B: one 128-bit load and one 128-bit store per nonzero.
// BLOCKED: thread t handles destination position ord[t] instead of t.  `ord` lists the destination
// positions grouped by the source block (2^block_log2 records) their record comes from, so at any
// time the whole grid gathers from one source window that stays in L2, and every 64-byte DRAM
// fetch is used completely; inside a group the destination positions ascend in long runs (the
// layouts' key orders are chosen for that, build.cu choose_key_order), so the stores stay whole sectors.
template <bool BLOCKED>
__global__ void __launch_bounds__(256) k_remap3(const uint4* __restrict__ in, const uint32_t* __restrict__ prev,
                                                const uint32_t* __restrict__ ord, const uint8_t* __restrict__ dflags,
                                                uint4* __restrict__ out, int64_t nnz, int64_t nnz_pad, FieldMap fm) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nnz_pad) return;
    const int64_t j = (BLOCKED && t < nnz) ? (int64_t)__ldcs(ord + t) : t;   // padding positions are handled in place
    const uint32_t src = BLOCKED ? __ldg(prev + (j < nnz ? j : nnz - 1)) : __ldcs(prev + (j < nnz ? j : nnz - 1));
    const uint4 r = __ldg(in + src);
    const uint32_t f[3] = {r.x & kKeyMask, r.y & kKeyMask, r.z & kKeyMask};
    uint32_t k[3];
#pragma unroll
    for (int l = 0; l < 3; ++l) k[l] = fm.src[l] == 0 ? f[0] : (fm.src[l] == 1 ? f[1] : f[2]);
    apply_run_flags<3>(k, dflags[j]);
    __stcs(out + j, make_uint4(k[0], k[1], k[2], j < nnz ? r.w : 0u));
}

template <int N, bool BLOCKED>
__global__ void __launch_bounds__(256) k_remap(const uint32_t* __restrict__ in, const uint32_t* __restrict__ prev,
                                               const uint32_t* __restrict__ ord, const uint8_t* __restrict__ dflags,
                                               uint32_t* __restrict__ out, int64_t nnz, int64_t nnz_pad, FieldMap fm) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nnz_pad) return;
    const int64_t j = (BLOCKED && t < nnz) ? (int64_t)__ldcs(ord + t) : t;
    const uint32_t* r = in + (size_t)__ldg(prev + (j < nnz ? j : nnz - 1)) * (N + 1);
    uint32_t k[N];
#pragma unroll
    for (int l = 0; l < N; ++l) k[l] = __ldg(r + fm.src[l]) & kKeyMask;
    apply_run_flags<N>(k, dflags[j]);
    uint32_t* o = out + (size_t)j * (N + 1);
#pragma unroll
    for (int l = 0; l < N; ++l) o[l] = k[l];
    o[N] = j < nnz ? __ldg(r + N) : 0u;
}

template <int N>
static void launch_remap_n(mttkrp_handle_s* h, int from, int to, unsigned grid, int64_t nnz_pad, const FieldMap& fm, cudaStream_t st) {
    const ModeMeta& mf = h->mode[from];
    const uint8_t* dflags = h->mode[to].lflags;
    if constexpr (N == 3) {
        if (mf.blocked) k_remap3<true><<<grid, 256, 0, st>>>((const uint4*)h->rec_cur, mf.next, mf.ord, dflags, (uint4*)h->rec_alt, h->nnz, nnz_pad, fm);
        else k_remap3<false><<<grid, 256, 0, st>>>((const uint4*)h->rec_cur, mf.next, mf.ord, dflags, (uint4*)h->rec_alt, h->nnz, nnz_pad, fm);
    } else {
        if (mf.blocked) k_remap<N, true><<<grid, 256, 0, st>>>(h->rec_cur, mf.next, mf.ord, dflags, h->rec_alt, h->nnz, nnz_pad, fm);
        else k_remap<N, false><<<grid, 256, 0, st>>>(h->rec_cur, mf.next, mf.ord, dflags, h->rec_alt, h->nnz, nnz_pad, fm);
    }
}

mttkrp_status_t launch_remap(mttkrp_handle_s* h, int from, cudaStream_t st) {
    const int N = h->N;
    const int to = (from + 1) % N;
    if (h->nnz > 0) {
        FieldMap fm;
        for (int l = 0; l < kMaxModes; ++l) fm.src[l] = 0;
        for (int l = 0; l < N; ++l) fm.src[l] = h->mode[from].pos[h->mode[to].order[l]];
        const int64_t nnz_pad = h->num_shards * (int64_t)h->shard_nnz;
        const unsigned grid = (unsigned)((nnz_pad + 255) / 256);
        TimedLaunch tl(h->timing, kClsRemap, st);
        switch (N) {
            case 2: launch_remap_n<2>(h, from, to, grid, nnz_pad, fm, st); break;
            case 3: launch_remap_n<3>(h, from, to, grid, nnz_pad, fm, st); break;
            case 4: launch_remap_n<4>(h, from, to, grid, nnz_pad, fm, st); break;
            case 5: launch_remap_n<5>(h, from, to, grid, nnz_pad, fm, st); break;
            case 6: launch_remap_n<6>(h, from, to, grid, nnz_pad, fm, st); break;
            case 7: launch_remap_n<7>(h, from, to, grid, nnz_pad, fm, st); break;
            case 8: launch_remap_n<8>(h, from, to, grid, nnz_pad, fm, st); break;
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

mttkrp_status_t launch_export(const mttkrp_handle_s* h, int32_t* idx, float* vals, cudaStream_t st) {
    if (h->nnz > 0) {
        PosArg pa;
        for (int m = 0; m < kMaxModes; ++m) pa.v[m] = h->mode[h->cur].pos[m];
        k_export<<<(unsigned)((h->nnz + 255) / 256), 256, 0, st>>>(h->rec_cur, h->nnz, h->N, pa, idx, vals);
        MK_CUDA(cudaGetLastError());
    }
    return MTTKRP_OK;
}

}  // namespace mk
