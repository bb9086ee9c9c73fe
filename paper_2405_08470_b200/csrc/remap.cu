// Dynamic tensor remapping (Alg. 3): T_out[next[k]] = T_in[k], where next[k] is
// the element's position in the layout of mode (d+1) mod N (its remap id).  Every
// element has a unique destination (Observation 1), so plain stores suffice.
// Records are role-ordered (sort keys major to minor, then the value), so the scatter also permutes
// the index fields from the source layout's key order to the destination's.
#include "common.cuh"

namespace mk {

struct FieldMap { int src[kMaxModes]; };   // out.field[l] = in.field[src[l]]

// 3-mode records are 16 B: one 128-bit load and one 128-bit store per nonzero.
__global__ void __launch_bounds__(256) k_remap3(const uint4* __restrict__ in, const uint32_t* __restrict__ next,
                                                uint4* __restrict__ out, int64_t nnz, FieldMap fm) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nnz) return;
    uint4 r = __ldcs(in + k);
    uint32_t dst = __ldcs(next + k);
    uint32_t f[3] = {r.x, r.y, r.z};
    uint4 o;
    o.x = fm.src[0] == 0 ? f[0] : (fm.src[0] == 1 ? f[1] : f[2]);
    o.y = fm.src[1] == 0 ? f[0] : (fm.src[1] == 1 ? f[1] : f[2]);
    o.z = fm.src[2] == 0 ? f[0] : (fm.src[2] == 1 ? f[1] : f[2]);
    o.w = r.w;
    out[dst] = o;
}

// Gather form: T_out[j] = T_in[prev[j]]: coalesced 16 B stores, random 16 B loads (no partial-sector
// writes, so no read-modify-write in DRAM).
__global__ void __launch_bounds__(256) k_remap3_gather(const uint4* __restrict__ in, const uint32_t* __restrict__ prev,
                                                       uint4* __restrict__ out, int64_t nnz, FieldMap fm) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nnz) return;
    uint32_t src = __ldcs(prev + j);
    uint4 r = __ldg(in + src);
    uint32_t f[3] = {r.x, r.y, r.z};
    uint4 o;
    o.x = fm.src[0] == 0 ? f[0] : (fm.src[0] == 1 ? f[1] : f[2]);
    o.y = fm.src[1] == 0 ? f[0] : (fm.src[1] == 1 ? f[1] : f[2]);
    o.z = fm.src[2] == 0 ? f[0] : (fm.src[2] == 1 ? f[1] : f[2]);
    o.w = r.w;
    __stcs(out + j, o);
}

template <int N>
__global__ void __launch_bounds__(256) k_remap_gather(const uint32_t* __restrict__ in, const uint32_t* __restrict__ prev,
                                                      uint32_t* __restrict__ out, int64_t nnz, FieldMap fm) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nnz) return;
    const uint32_t* r = in + (size_t)__ldcs(prev + j) * (N + 1);
    uint32_t* o = out + (size_t)j * (N + 1);
#pragma unroll
    for (int l = 0; l < N; ++l) o[l] = __ldg(r + fm.src[l]);
    o[N] = __ldg(r + N);
}

template <int N>
__global__ void __launch_bounds__(256) k_remap(const uint32_t* __restrict__ in, const uint32_t* __restrict__ next,
                                               uint32_t* __restrict__ out, int64_t nnz, FieldMap fm) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nnz) return;
    const uint32_t* r = in + (size_t)k * (N + 1);
    uint32_t* o = out + (size_t)__ldcs(next + k) * (N + 1);
#pragma unroll
    for (int l = 0; l < N; ++l) o[l] = r[fm.src[l]];
    o[N] = r[N];
}

mttkrp_status_t launch_remap(mttkrp_handle_s* h, int from, cudaStream_t st) {
    const int N = h->N;
    const int to = (from + 1) % N;
    if (h->nnz > 0) {
        FieldMap fm;
        for (int l = 0; l < kMaxModes; ++l) fm.src[l] = 0;
        for (int l = 0; l < N; ++l) fm.src[l] = h->mode[from].pos[h->mode[to].order[l]];
        const unsigned grid = (unsigned)((h->nnz + 255) / 256);
        const uint32_t* next = h->mode[from].next;
        TimedLaunch tl(h->timing, kClsRemap, st);
        if (h->remap_gather) {
            switch (N) {
                case 2: k_remap_gather<2><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
                case 3: k_remap3_gather<<<grid, 256, 0, st>>>((const uint4*)h->rec_cur, next, (uint4*)h->rec_alt, h->nnz, fm); break;
                case 4: k_remap_gather<4><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
                case 5: k_remap_gather<5><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
                case 6: k_remap_gather<6><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
                case 7: k_remap_gather<7><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
                case 8: k_remap_gather<8><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
                default: set_error("remap: unsupported nmodes %d", N); return MTTKRP_EUNSUPPORTED;
            }
        } else
        switch (N) {
            case 2: k_remap<2><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
            case 3: k_remap3<<<grid, 256, 0, st>>>((const uint4*)h->rec_cur, next, (uint4*)h->rec_alt, h->nnz, fm); break;
            case 4: k_remap<4><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
            case 5: k_remap<5><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
            case 6: k_remap<6><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
            case 7: k_remap<7><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
            case 8: k_remap<8><<<grid, 256, 0, st>>>(h->rec_cur, next, h->rec_alt, h->nnz, fm); break;
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

// Carries the original-position array from one layout to the next:
// scatter map: out[map[k]] = in[k]; gather map: out[j] = in[map[j]].
__global__ void k_perm_step(const uint32_t* __restrict__ map, int gather, const uint32_t* __restrict__ in,
                            uint32_t* __restrict__ out, int64_t nnz) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nnz) return;
    if (gather) out[k] = in[map[k]];
    else out[map[k]] = in[k];
}

mttkrp_status_t launch_perm_step(const uint32_t* map, int gather, const uint32_t* in, uint32_t* out, int64_t nnz, cudaStream_t st) {
    if (nnz > 0) {
        k_perm_step<<<(unsigned)((nnz + 255) / 256), 256, 0, st>>>(map, gather, in, out, nnz);
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
    for (int m = 0; m < N; ++m) idx[(size_t)m * nnz + k] = (int32_t)r[pos.v[m]];
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
