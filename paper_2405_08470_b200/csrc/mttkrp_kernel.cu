// spMTTKRP for one mode on the mode-d layout (Alg. 2 "Elementwise Computation", PAPER.md:197-217;
// Alg. 4 thread-block mapping, as function only; the mapping here is this
// library's own).
//
// Layout: records sorted by the key tuple (k_0 = i_d, k_1, ..., k_{N-1}); record = N int32 keys in
// that order + fp32 value.  A thread block owns one shard = shard_nnz consecutive records
// (equal-nnz shards).  Inside the block a GROUP of R/4 lanes (one float4 of the rank dimension per
// lane) walks a contiguous chunk of the shard one nonzero at a time:
//   l(r) = val * prod_w A_w[i_w, r]         (Alg. 2 lines 8-13)
//   Y_d[i_d, r] += l(r)                     (Alg. 2 lines 14-15)
// Because the chunk is sorted, the products are nested sums (a CSF-style factoring of the same
// expression):  Y[k_0] = sum_{k_1} A[k_1] * ( sum_{k_2} A[k_2] * ( ... sum_{k_{N-1}} val * A[k_{N-1}] ) ),
// so a factor row is gathered once per run of equal key prefix rather than once per nonzero.
// Rows that begin and end inside a chunk are stored with plain stores by their only owner
// (Observation 2: no global atomics).  The first/last partial rows of each chunk
// are merged in shared memory by warp 0; a row that spans shards leaves one partial per shard in the
// carry buffer and is summed, in fixed order, by k_fixup.  Rows with no nonzero are zeroed by
// k_zero_rows from the precomputed list, so `out` is fully overwritten without a memset.
#include <algorithm>
#include "common.cuh"

namespace mk {

template <int N>
struct KernelArgs {
    const uint32_t* rec;
    int64_t nnz;
    int shard_nnz;
    const float* fac[N];     // fac[l] = factor of the mode at key level l (fac[0] unused)
    float* out;
    float* carry;            // [2*num_shards][R]
};

__device__ __forceinline__ float4 ld_row(const float* __restrict__ A, uint32_t row, int R, int sub) {
    return __ldg(reinterpret_cast<const float4*>(A + (size_t)row * R) + sub);
}
__device__ __forceinline__ void fma4(float4& acc, const float4& a, const float4& b) {
    acc.x = fmaf(a.x, b.x, acc.x);
    acc.y = fmaf(a.y, b.y, acc.y);
    acc.z = fmaf(a.z, b.z, acc.z);
    acc.w = fmaf(a.w, b.w, acc.w);
}
__device__ __forceinline__ void fma4s(float4& acc, float s, const float4& b) {
    acc.x = fmaf(s, b.x, acc.x);
    acc.y = fmaf(s, b.y, acc.y);
    acc.z = fmaf(s, b.z, acc.z);
    acc.w = fmaf(s, b.w, acc.w);
}

template <int N>
struct Rec {
    uint32_t k[N];
    float val;
};

template <int N>
__device__ __forceinline__ Rec<N> load_rec(const uint32_t* __restrict__ rec, int64_t pos) {
    Rec<N> r;
    const uint32_t* p = rec + (size_t)pos * (N + 1);
    if constexpr (N == 3) {
        uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
        r.k[0] = v.x; r.k[1] = v.y; r.k[2] = v.z; r.val = __uint_as_float(v.w);
    } else if constexpr (N == 7) {
        uint4 a = __ldg(reinterpret_cast<const uint4*>(p));
        uint4 b = __ldg(reinterpret_cast<const uint4*>(p) + 1);
        r.k[0] = a.x; r.k[1] = a.y; r.k[2] = a.z; r.k[3] = a.w;
        r.k[4] = b.x; r.k[5] = b.y; r.k[6] = b.z; r.val = __uint_as_float(b.w);
    } else if constexpr ((N + 1) % 2 == 0) {
        uint32_t w[N + 1];
#pragma unroll
        for (int j = 0; j < (N + 1) / 2; ++j) {
            uint2 v = __ldg(reinterpret_cast<const uint2*>(p) + j);
            w[2 * j] = v.x; w[2 * j + 1] = v.y;
        }
#pragma unroll
        for (int j = 0; j < N; ++j) r.k[j] = w[j];
        r.val = __uint_as_float(w[N]);
    } else {
#pragma unroll
        for (int j = 0; j < N; ++j) r.k[j] = __ldg(p + j);
        r.val = __uint_as_float(__ldg(p + N));
    }
    return r;
}

template <int N, int R>
__global__ void __launch_bounds__(kBlockThreads) k_mttkrp(const KernelArgs<N> a) {
    constexpr int LPN = R / 4;                   // lanes per nonzero
    constexpr int NPW = 32 / LPN;                // groups per warp
    constexpr int G = (kBlockThreads / 32) * NPW;   // groups per block
    constexpr int NL = N - 1;                    // accumulator levels t[0..NL-1]
    __shared__ __align__(16) float ent_vec[2 * G][R];
    __shared__ int ent_row[2 * G];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gi = warp * NPW + lane / LPN;
    const int sub = lane % LPN;
    const int64_t shard = blockIdx.x;
    const int64_t s_begin = shard * (int64_t)a.shard_nnz;
    const int64_t s_end = min(s_begin + a.shard_nnz, a.nnz);
    const int C = a.shard_nnz / G;
    const int64_t c_begin = min(s_begin + (int64_t)gi * C, s_end);
    const int64_t c_end = min(c_begin + C, s_end);

    uint32_t key[NL];
    float4 t[NL];
    float4 rowv[NL];                             // rowv[l] = A_{level l}[key[l]] for l >= 1
#pragma unroll
    for (int l = 0; l < NL; ++l) {
        key[l] = 0xffffffffu;
        t[l] = make_float4(0.f, 0.f, 0.f, 0.f);
        rowv[l] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    int seg = 0;                                 // output-row segments finished so far in this chunk
    float* const entF = &ent_vec[2 * gi][sub * 4];
    float* const entL = &ent_vec[2 * gi + 1][sub * 4];

    if (c_begin < c_end) {
        Rec<N> cur = load_rec<N>(a.rec, c_begin);
        for (int64_t pos = c_begin; pos < c_end; ++pos) {
            Rec<N> nxt = cur;
            if (pos + 1 < c_end) nxt = load_rec<N>(a.rec, pos + 1);
            const float4 alast = ld_row(a.fac[N - 1], cur.k[N - 1], R, sub);
            int c = NL;                          // first key level that differs from the running prefix
#pragma unroll
            for (int l = NL - 1; l >= 0; --l)
                if (cur.k[l] != key[l]) c = l;
            if (c < NL) {
                // close the finished runs, innermost first: t[l-1] += A[key[l]] * t[l]
#pragma unroll
                for (int l = NL - 1; l >= 1; --l) {
                    if (l >= c) {
                        fma4(t[l - 1], rowv[l], t[l]);
                        t[l] = make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                }
                if (c == 0) {
                    if (key[0] != 0xffffffffu) {
                        float* dst = (seg == 0) ? entF : a.out + (size_t)key[0] * R + sub * 4;
                        *reinterpret_cast<float4*>(dst) = t[0];
                        if (seg == 0 && sub == 0) ent_row[2 * gi] = (int)key[0];
                        ++seg;
                    }
                    t[0] = make_float4(0.f, 0.f, 0.f, 0.f);
                }
#pragma unroll
                for (int l = 0; l < NL; ++l) {
                    if (l >= c) {
                        key[l] = cur.k[l];
                        if (l >= 1) rowv[l] = ld_row(a.fac[l], key[l], R, sub);
                    }
                }
            }
            fma4s(t[NL - 1], cur.val, alast);
            cur = nxt;
        }
#pragma unroll
        for (int l = NL - 1; l >= 1; --l) fma4(t[l - 1], rowv[l], t[l]);
        float* dst = (seg == 0) ? entF : entL;
        *reinterpret_cast<float4*>(dst) = t[0];
        if (sub == 0) {
            ent_row[2 * gi + (seg == 0 ? 0 : 1)] = (int)key[0];
            if (seg == 0) ent_row[2 * gi + 1] = -1;
        }
    } else if (sub == 0) {
        ent_row[2 * gi] = -1;
        ent_row[2 * gi + 1] = -1;
    }
    __syncthreads();

    // Merge the chunk-boundary partials in order; runs of equal row are adjacent.
    if (warp == 0 && s_begin < s_end) {
        const uint32_t first_row = __ldg(a.rec + (size_t)s_begin * (N + 1));
        const uint32_t last_row = __ldg(a.rec + (size_t)(s_end - 1) * (N + 1));
        const bool head_shared = s_begin > 0 && __ldg(a.rec + (size_t)(s_begin - 1) * (N + 1)) == first_row;
        const bool tail_shared = s_end < a.nnz && __ldg(a.rec + (size_t)s_end * (N + 1)) == last_row;
        constexpr int CPL = (R + 31) / 32;       // columns per lane
        float acc[CPL];
#pragma unroll
        for (int j = 0; j < CPL; ++j) acc[j] = 0.f;
        int cur_row = -1;
        auto emit = [&](int row) {
            float* dst;
            if ((uint32_t)row == first_row && head_shared) dst = a.carry + (size_t)(2 * shard) * R;
            else if ((uint32_t)row == last_row && tail_shared) dst = a.carry + (size_t)(2 * shard + 1) * R;
            else dst = a.out + (size_t)row * R;
#pragma unroll
            for (int j = 0; j < CPL; ++j) {
                int col = lane + 32 * j;
                if (col < R) dst[col] = acc[j];
            }
        };
        for (int e = 0; e < 2 * G; ++e) {
            const int r = ent_row[e];
            if (r < 0) continue;
            if (r != cur_row) {
                if (cur_row >= 0) emit(cur_row);
                cur_row = r;
#pragma unroll
                for (int j = 0; j < CPL; ++j) acc[j] = 0.f;
            }
#pragma unroll
            for (int j = 0; j < CPL; ++j) {
                int col = lane + 32 * j;
                if (col < R) acc[j] += ent_vec[e][col];
            }
        }
        if (cur_row >= 0) emit(cur_row);
    }
}

// Y[row] = carry[2*s+1] + sum_{j=s+1..t} carry[2*j] for every split row (s, t, row), fixed order.
template <int R>
__global__ void __launch_bounds__(128) k_fixup(const uint32_t* __restrict__ chains, const float* __restrict__ carry,
                                               float* __restrict__ out) {
    constexpr int LPN = R / 4;
    constexpr int G = 128 / LPN;
    __shared__ __align__(16) float part[G][R];
    const uint32_t s = chains[3 * (size_t)blockIdx.x], t = chains[3 * (size_t)blockIdx.x + 1];
    const uint32_t row = chains[3 * (size_t)blockIdx.x + 2];
    const int g = threadIdx.x / LPN, sub = threadIdx.x % LPN;
    const int len = (int)(t - s) + 1;            // entries: j = 0 -> slot 2s+1, j >= 1 -> slot 2(s+j)
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int j = g; j < len; j += G) {
        const size_t slot = (j == 0) ? (size_t)2 * s + 1 : (size_t)2 * (s + j);
        const float4 v = *(reinterpret_cast<const float4*>(carry + slot * R) + sub);
        acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    *reinterpret_cast<float4*>(&part[g][sub * 4]) = acc;
    __syncthreads();
    if (threadIdx.x < R) {
        float sum = 0.f;
        const int used = len < G ? len : G;
        for (int q = 0; q < used; ++q) sum += part[q][threadIdx.x];
        out[(size_t)row * R + threadIdx.x] = sum;
    }
}

template <int R>
__global__ void __launch_bounds__(256) k_zero_rows(const uint32_t* __restrict__ rows, int64_t n, float* __restrict__ out) {
    constexpr int LPN = R / 4;
    const int64_t gid = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / LPN;
    const int sub = threadIdx.x % LPN;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x / LPN;
    for (int64_t i = gid; i < n; i += stride)
        *(reinterpret_cast<float4*>(out + (size_t)rows[i] * R) + sub) = make_float4(0.f, 0.f, 0.f, 0.f);
}

template <int N, int R>
static mttkrp_status_t launch_nr(const mttkrp_handle_s* h, int d, const float* const* factors, float* out,
                                 cudaStream_t st) {
    const ModeMeta& mm = h->mode[d];
    if (mm.n_empty > 0) {
        const int64_t groups = mm.n_empty;
        const int64_t threads = groups * (R / 4);
        const unsigned grid = (unsigned)std::min<int64_t>((threads + 255) / 256, 148 * 16);
        TimedLaunch tl(h->timing, kClsZero, st);
        k_zero_rows<R><<<grid, 256, 0, st>>>(mm.empty_rows, mm.n_empty, out);
    }
    if (h->num_shards > 0) {
        KernelArgs<N> a;
        a.rec = h->rec_cur;
        a.nnz = h->nnz;
        a.shard_nnz = h->shard_nnz;
        a.fac[0] = nullptr;
        for (int l = 1; l < N; ++l) a.fac[l] = factors[mm.order[l]];
        a.out = out;
        a.carry = h->carry;
        {
            TimedLaunch tl(h->timing, kClsMttkrp, st);
            k_mttkrp<N, R><<<(unsigned)h->num_shards, kBlockThreads, 0, st>>>(a);
        }
        if (mm.n_chains > 0) {
            TimedLaunch tl(h->timing, kClsFixup, st);
            k_fixup<R><<<(unsigned)mm.n_chains, 128, 0, st>>>(mm.chains, h->carry, out);
        }
    }
    MK_CUDA(cudaGetLastError());
    return MTTKRP_OK;
}

template <int N>
static mttkrp_status_t launch_n(const mttkrp_handle_s* h, int d, const float* const* factors, int R, float* out,
                                cudaStream_t st) {
    switch (R) {
        case 8: return launch_nr<N, 8>(h, d, factors, out, st);
        case 16: return launch_nr<N, 16>(h, d, factors, out, st);
        case 32: return launch_nr<N, 32>(h, d, factors, out, st);
        case 64: return launch_nr<N, 64>(h, d, factors, out, st);
    }
    set_error("unsupported rank %d (8, 16, 32, 64)", R);
    return MTTKRP_EUNSUPPORTED;
}

mttkrp_status_t launch_mttkrp(const mttkrp_handle_s* h, int d, const float* const* factors, int R, float* out,
                              cudaStream_t st) {
    switch (h->N) {
        case 2: return launch_n<2>(h, d, factors, R, out, st);
        case 3: return launch_n<3>(h, d, factors, R, out, st);
        case 4: return launch_n<4>(h, d, factors, R, out, st);
        case 5: return launch_n<5>(h, d, factors, R, out, st);
        case 6: return launch_n<6>(h, d, factors, R, out, st);
        case 7: return launch_n<7>(h, d, factors, R, out, st);
        case 8: return launch_n<8>(h, d, factors, R, out, st);
    }
    set_error("unsupported nmodes %d", h->N);
    return MTTKRP_EUNSUPPORTED;
}

}  // namespace mk
