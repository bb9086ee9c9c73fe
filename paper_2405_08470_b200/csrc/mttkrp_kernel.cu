// spMTTKRP for one mode on the mode-d layout (Alg. 2 "Elementwise Computation", PAPER.md:197-217;
// Alg. 4 thread-block mapping, as function only; the mapping here is this
// library's own, made for sm_100a).
//
// Layout: records sorted by the key tuple (k_0 = i_d, k_1, ..., k_{N-1}); record = N uint32 keys in
// that order + fp32 value, or (N >= 4, PACKED) 16 bytes with the keys bit-packed (common.cuh PackDesc).
// The record carries the run-end flags that the format builder and the remap pass derived from the
// sorted order (bit 31 of the key words / top bits of w2, common.cuh), so it is self-contained: the hot
// loop has no look-ahead compare.
// A thread block owns one shard = shard_nnz consecutive records (equal-nnz shards).  Inside the
// block a GROUP of R/V lanes (V = 4 rank columns per lane, one 128-bit LDG per factor row per lane:
// a warp instruction then covers whole 128-byte lines, one L1 wavefront each) walks a contiguous
// chunk of the shard one nonzero at a time:
//   l(r) = val * prod_w A_w[i_w, r]         (Alg. 2 lines 8-13)
//   Y_d[i_d, r] += l(r)                     (Alg. 2 lines 14-15)
// Because the chunk is sorted, the products are nested sums (a CSF-style factoring of the same
// expression):  Y[k_0] = sum_{k_1} A[k_1] * ( sum_{k_2} A[k_2] * ( ... sum_{k_{N-1}} val * A[k_{N-1}] ) ),
// so the row of level l is gathered once per run of equal (k_0..k_l), at the END of the run.
//
// Pipeline per warp: records are staged into a shared-memory ring with cp.async (stages of K
// records per group, interleaved by group so one LDS.128 serves all groups without bank conflicts).
// D steps ahead of the arithmetic the group reads its record from the ring and issues the
// factor-row gathers for that step into rotating registers.  The arithmetic is packed fp32x2 FMA.
// The kernel is bound by the L1 data pipe (one wavefront per gathered line), so every other use of
// that pipe is kept minimal: one cp.async and one LDS per record.
//
// Rows that begin and end inside a chunk are stored with plain stores by their only owner
// (Observation 2: no global atomics).  The first/last partial rows of each chunk
// are merged in shared memory, first per warp, then per block; a row that spans shards leaves one
// partial per shard in the carry buffer and is summed, in fixed order, by k_fixup.  Rows with no
// nonzero are zeroed by k_zero_rows from the precomputed list, so `out` is fully overwritten
// without a memset.
#include <algorithm>
#include <type_traits>
#include "common.cuh"

namespace mk {

template <int N>
struct KernelArgs {
    const uint32_t* rec;     // padded to num_shards * shard_nnz records
    int64_t nnz;             // padded record count
    int shard_nnz;
    const float* fac[N];     // fac[l] = factor of the mode at key level l (fac[0] unused)
    float* out;
    float* carry;            // [2*num_shards][R]
    uint32_t kmask[N];       // packed records (common.cuh PackDesc): mask and bit offset of the key of level l;
    int32_t koff[N];         // kmask[0] also masks word 0 of unpacked records (all ones)
};

// ---- small PTX helpers ------------------------------------------------------------------------
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;"
        : "=l"(d)
        : "l"(*reinterpret_cast<unsigned long long*>(&a)), "l"(*reinterpret_cast<unsigned long long*>(&b)),
          "l"(*reinterpret_cast<unsigned long long*>(&c)));
    return *reinterpret_cast<float2*>(&d);
}
__device__ __forceinline__ float2 splat2(float s) {
    unsigned long long d;
    asm("mov.b64 %0, {%1, %1};" : "=l"(d) : "f"(s));
    return *reinterpret_cast<float2*>(&d);
}

template <int V>
struct Vec {                 // V rank columns of one lane, as fp32 pairs
    float2 p[V / 2];
};

template <int V>
__device__ __forceinline__ Vec<V> vzero() {
    Vec<V> r;
#pragma unroll
    for (int i = 0; i < V / 2; ++i) r.p[i] = make_float2(0.f, 0.f);
    return r;
}

#ifndef MK_L2HINT        // 1: the record stream is read with an L2 evict-first policy, so that it does not push the
#define MK_L2HINT 1      //    factor rows (the data that is re-used) out of L2 (measured: -2 % on configs[1], -1 % on
                         //    configs[2]; an evict-last hint on the factor rows themselves was 10 % slower)
#endif
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// One lane's V columns of a factor row (read-only path; 128-bit or 256-bit load).
// `base` = factor matrix (uniform), `word` = row index with bit 31 (run-end flag) ignored, `sub` = this
// lane's slot inside the row.  The element offset (row * R/V + sub) is formed in 32 bits - the shift
// drops the flag bit - and scaled by one 32x32->64 multiply-add on the uniform base, so a row address
// costs two instructions and no per-lane pointer registers.  Needs dims[m] < 2^28 (api.cu check_shape).
template <int V, int R>
__device__ __forceinline__ Vec<V> ld_row(const float* __restrict__ base, uint32_t word, uint32_t sub) {
    constexpr int SH = (R / V == 16) ? 4 : (R / V == 8) ? 3 : (R / V == 4) ? 2 : 1;      // log2(lanes per row)
    const uint32_t off = (word << SH) + sub;
    Vec<V> r;
    if constexpr (V == 8) {
        const float* p = base + (size_t)off * 8;
        asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=f"(r.p[0].x), "=f"(r.p[0].y), "=f"(r.p[1].x), "=f"(r.p[1].y), "=f"(r.p[2].x), "=f"(r.p[2].y),
                       "=f"(r.p[3].x), "=f"(r.p[3].y)
                     : "l"(p));
    } else {
        const float4 v = __ldg(reinterpret_cast<const float4*>(base) + off);
        r.p[0] = make_float2(v.x, v.y);
        r.p[1] = make_float2(v.z, v.w);
    }
    return r;
}
// acc += a * b (elementwise), acc += s * b
template <int V>
__device__ __forceinline__ void vfma(Vec<V>& acc, const Vec<V>& a, const Vec<V>& b) {
#pragma unroll
    for (int i = 0; i < V / 2; ++i) acc.p[i] = ffma2(a.p[i], b.p[i], acc.p[i]);
}
template <int V>
__device__ __forceinline__ void vfmas(Vec<V>& acc, float s, const Vec<V>& b) {
    const float2 ss = splat2(s);
#pragma unroll
    for (int i = 0; i < V / 2; ++i) acc.p[i] = ffma2(ss, b.p[i], acc.p[i]);
}
template <int V>
__device__ __forceinline__ void vstore(float* dst, const Vec<V>& v) {
#pragma unroll
    for (int i = 0; i < V / 4; ++i)
        *reinterpret_cast<float4*>(dst + 4 * i) = make_float4(v.p[2 * i].x, v.p[2 * i].y, v.p[2 * i + 1].x, v.p[2 * i + 1].y);
}

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, uint64_t policy) {
#if MK_L2HINT
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "l"(policy) : "memory");
#else
    (void)policy;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
#endif
}
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPEND>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NPEND) : "memory"); }

// ---- compile-time geometry ---------------------------------------------------------------------
#ifndef MK_V8
#define MK_V8 0          // 1: 8 columns per lane (256-bit gathers); measured 1.4 L1 wavefronts per 128-byte line
#endif                   //    against 1.0 for 128-bit gathers
#ifndef MK_D
#define MK_D 2
#endif
#ifndef MK_STAGES
#define MK_STAGES 3
#endif
#ifndef MK_MINB          // resident blocks per SM the register allocation must allow; 0 = per-N default below.
#define MK_MINB 0        // Measured on B200 (configs[1], configs[2]): occupancy beats deeper look-ahead.
#endif
template <int N, int R, bool DEEP, bool PACKED>
struct Geo {
    static constexpr int V = (MK_V8 && R >= 16) ? 8 : 4; // rank columns per lane
    static constexpr int LPN = R / V;                    // lanes per nonzero (group size)
    static constexpr int NPW = 32 / LPN;                 // groups per warp
    static constexpr int WARPS = kBlockThreads / 32;
    static constexpr int G = WARPS * NPW;                // groups per block
    static constexpr int RECW = PACKED ? 4 : N + 1;      // record words
    static constexpr int SLOTW = (RECW + 3) / 4 * 4;     // ring slot words (16-byte multiple)
    static constexpr int K = (NPW * SLOTW <= 32) ? 8 : 4;  // records per group per ring stage
    static constexpr int STAGES = MK_STAGES;             // round r computing, r+1 landed, the rest in flight
    // gather look-ahead, in steps (K % D == 0).  DEEP: twice the look-ahead at one block per SM less, for
    // factor matrices that do not fit L2 (every gather that misses is a random HBM access).
    static constexpr int D0 = (DEEP && N <= 3) ? 2 * MK_D : MK_D;
    static constexpr int D = (D0 < K) ? D0 : K / 2;
    static constexpr int RING_WORDS = STAGES * K * NPW * SLOTW;        // per warp
    static constexpr int ENT_WORDS = 2 * NPW * R;                       // per warp: first/last partial rows
    static constexpr int WARP_WORDS = RING_WORDS > ENT_WORDS ? RING_WORDS : ENT_WORDS;
    static constexpr int NL = N - 1;                     // accumulator levels t[0..NL-1]
    static constexpr int MINB = MK_MINB ? MK_MINB : (N <= 3 ? (DEEP ? 4 : 5) : (N == 4 ? 4 : 3));
    static constexpr int SMEM_BYTES = 4 * (WARPS * WARP_WORDS + WARPS * NPW * R + 2 * WARPS * R + WARPS * 2 * NPW + 2 * WARPS);
};

// Sequential merge of partial rows (rows[e] < 0 = unused).  Runs of equal row id are adjacent.
// emit(row, acc, is_first_run, is_last_run): lane c holds columns c, c+32.
template <int R, class Emit>
__device__ __forceinline__ void merge_runs(const int* rows, const float* vecs, int n, int lane, Emit emit) {
    constexpr int CPL = (R + 31) / 32;
    float acc[CPL];
#pragma unroll
    for (int j = 0; j < CPL; ++j) acc[j] = 0.f;
    int cur_row = -1, run = 0;
    for (int e = 0; e < n; ++e) {
        const int r = rows[e];
        if (r < 0) continue;
        if (r != cur_row) {
            if (cur_row >= 0) { emit(cur_row, acc, run == 0, false); ++run; }
            cur_row = r;
#pragma unroll
            for (int j = 0; j < CPL; ++j) acc[j] = 0.f;
        }
#pragma unroll
        for (int j = 0; j < CPL; ++j) {
            const int col = lane + 32 * j;
            if (col < R) acc[j] += vecs[(size_t)e * R + col];
        }
    }
    if (cur_row >= 0) emit(cur_row, acc, run == 0, true);
}

template <int N, int R, bool DEEP, bool PACKED>
__global__ void __launch_bounds__(kBlockThreads, Geo<N, R, DEEP, PACKED>::MINB) k_mttkrp(const KernelArgs<N> a) {
    using Ge = Geo<N, R, DEEP, PACKED>;
    constexpr int V = Ge::V, LPN = Ge::LPN, NPW = Ge::NPW, WARPS = Ge::WARPS, G = Ge::G, K = Ge::K, D = Ge::D;
    constexpr int STAGES = Ge::STAGES, RECW = Ge::RECW, SLOTW = Ge::SLOTW, NL = Ge::NL;
    constexpr int ROWW = NPW * SLOTW;                     // ring words between consecutive records of a group
    constexpr int STAGEW = K * ROWW;                      // ring words per stage
    // cp.async piece: the widest power of two (4, 8 or 16 bytes) dividing the record
    constexpr int PW = RECW % 4 == 0 ? 4 : (RECW % 2 == 0 ? 2 : 1);
    constexpr int PPR = RECW / PW;                        // pieces per record
    constexpr int NPIECE = (K * PPR + LPN - 1) / LPN;     // pieces per lane per round
    constexpr int AHEAD = STAGES - 1;                     // rounds issued ahead of the one being computed
    static_assert(K % D == 0 && D < K && STAGES >= 3, "geometry");

    extern __shared__ uint4 smem_raw[];
    // carve-up (Geo::SMEM_BYTES): record rings (later the groups' last partial rows) | the groups'
    // first partial rows | the warps' first/last partial rows | row ids
    uint32_t (*s_warp)[Ge::WARP_WORDS] = reinterpret_cast<uint32_t (*)[Ge::WARP_WORDS]>(smem_raw);
    float (*s_first)[NPW][R] = reinterpret_cast<float (*)[NPW][R]>(&s_warp[WARPS][0]);
    float (*s_wvec)[R] = reinterpret_cast<float (*)[R]>(&s_first[WARPS][0][0]);
    int (*s_erow)[2 * NPW] = reinterpret_cast<int (*)[2 * NPW]>(&s_wvec[2 * WARPS][0]);
    int* s_wrow = &s_erow[WARPS][0];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane / LPN, sub = lane % LPN;
    const int64_t shard = blockIdx.x;
    // The record array is padded to a whole number of shards (value 0, keys of the last nonzero),
    // so every chunk holds exactly C records and the loop needs no bounds checks.
    const int64_t s_begin = shard * (int64_t)a.shard_nnz;
    const int64_t s_end = s_begin + a.shard_nnz;
    const int C = a.shard_nnz / G;                        // records per group; a multiple of K, > D
    const int nrounds = C / K;
    const int64_t cb = s_begin + (int64_t)(warp * NPW + g) * C;         // this group's first position
    const uint32_t* const grec = a.rec + (size_t)cb * RECW;

    uint32_t* const ring = &s_warp[warp][0];
    const uint32_t* const ring_g = ring + g * SLOTW;      // this group's column of the ring
    const uint32_t ring_gs = (uint32_t)__cvta_generic_to_shared(ring_g);

    const uint64_t rec_policy = l2_policy_evict_first();
    auto issue_round = [&](int r) {
        if (r < nrounds) {
            const uint32_t* src = grec + (size_t)r * (K * RECW);
            const uint32_t dst = ring_gs + 4u * (uint32_t)((r % STAGES) * STAGEW);
#pragma unroll
            for (int i = 0; i < NPIECE; ++i) {
                const int p = sub + i * LPN;
                if (p < K * PPR) {
                    const int jj = p / PPR, q = p % PPR;
                    const uint32_t d2 = dst + 4u * (uint32_t)(jj * ROWW + q * PW);
                    if constexpr (PW == 4) cp_async16(d2, src + jj * RECW + q * PW, rec_policy);
                    else if constexpr (PW == 2) cp_async8(d2, src + jj * RECW + q * PW);
                    else cp_async4(d2, src + jj * RECW + q * PW);
                }
            }
        }
        cp_async_commit();
    };
    auto read_slot = [&](const uint32_t* slot, uint32_t* w) {
        const uint4* p = reinterpret_cast<const uint4*>(slot);
#pragma unroll
        for (int i = 0; i < SLOTW / 4; ++i) {
            const uint4 v = p[i];
            w[4 * i] = v.x; w[4 * i + 1] = v.y; w[4 * i + 2] = v.z; w[4 * i + 3] = v.w;
        }
    };

    Vec<V> t[NL];                                         // t[0] = output row accumulator
#pragma unroll
    for (int l = 0; l < NL; ++l) t[l] = vzero<V>();
    Vec<V> al[D];                                         // last-level rows for the D steps in flight
    Vec<V> rb[NL][D];                                     // rb[l][slot]: row of level l, gathered at the end of its run
    float val[D];
    uint32_t fl[D];                                       // bit l: the run of level l ends at this step
    int seg = 0;                                          // output-row segments finished in this chunk

    // Issue the gathers of one step whose record sits at `slot`.  The record carries its run-end
    // flags (common.cuh).  The chunk's last record closes every inner run and leaves the output row
    // open: it is finished by the epilogue, which knows whether the row continues in the next chunk.
    auto prefetch = [&](const uint32_t* slot, int s, bool chunk_last) {
        uint32_t w[SLOTW];
        read_slot(slot, w);
        if constexpr (PACKED) {                           // {w0, w1, w2 = flags | last key, val}
            uint32_t f = w[2] >> (32 - (N - 1));
            if (chunk_last) f = (f | ((1u << NL) - 2u)) & ~1u;
            al[s] = ld_row<V, R>(a.fac[N - 1], w[2] & a.kmask[N - 1], sub);
#pragma unroll
            for (int l = 1; l < NL; ++l)
                if (f & (1u << l)) rb[l][s] = ld_row<V, R>(a.fac[l], pk_get(w[0], w[1], a.koff[l], a.kmask[l]), sub);
            val[s] = __uint_as_float(w[3]);
            fl[s] = f;
        } else {
            if (chunk_last) {
#pragma unroll
                for (int l = 1; l < NL; ++l) w[l] |= kFlag;
                w[N - 1] &= kKeyMask;
            }
            al[s] = ld_row<V, R>(a.fac[N - 1], w[N - 1], sub);
            uint32_t f = w[N - 1] >> 31;
#pragma unroll
            for (int l = 1; l < NL; ++l) {
                if (w[l] & kFlag) rb[l][s] = ld_row<V, R>(a.fac[l], w[l], sub);
                f |= (w[l] >> 31) << l;
            }
            val[s] = __uint_as_float(w[N]);
            fl[s] = f;
        }
    };
    // Arithmetic of one step (its record sits at `slot`).
    auto compute = [&](const uint32_t* slot, int s) {
        const uint32_t e = fl[s];
        vfmas<V>(t[NL - 1], val[s], al[s]);
#pragma unroll
        for (int l = NL - 1; l >= 1; --l) {
            if (e & (1u << l)) {
                vfma<V>(t[l - 1], rb[l][s], t[l]);
                t[l] = vzero<V>();
            }
        }
        if (e & 1u) {                                     // an output row ends inside the chunk
            const uint32_t row = slot[0] & a.kmask[0];
            if (seg == 0) {
                vstore<V>(&s_first[warp][g][sub * V], t[0]);
                if (sub == 0) s_erow[warp][2 * g] = (int)row;
            } else {
                vstore<V>(a.out + (size_t)row * R + sub * V, t[0]);
            }
            ++seg;
            t[0] = vzero<V>();
        }
    };

    // ---- prologue: rounds 0..AHEAD-1 in flight, round 0 landed ----------------------------------------
#pragma unroll
    for (int r = 0; r < AHEAD; ++r) issue_round(r);
    cp_async_wait<AHEAD - 1>();                           // round 0 has landed
    __syncwarp();
#pragma unroll
    for (int i = 0; i < D; ++i) prefetch(ring_g + i * ROWW, i, false);
    for (int r = 0; r < nrounds; ++r) {
        issue_round(r + AHEAD);                           // reuses the stage of round r-1
        cp_async_wait<AHEAD - 1>();                       // rounds <= r+1 have landed
        __syncwarp();
        const uint32_t* cs = ring_g + (r % STAGES) * STAGEW;            // this round's stage
        const uint32_t* ns = ring_g + ((r + 1) % STAGES) * STAGEW;      // next round's stage
        const bool more = r + 1 < nrounds;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            compute(cs + i * ROWW, i % D);
            if (i + D < K) prefetch(cs + (i + D) * ROWW, i % D, (i + D == K - 1) && !more);
            else if (more) prefetch(ns + (i + D - K) * ROWW, i % D, false);
        }
        __syncwarp();                                     // everyone is done with round r's stage
    }
    cp_async_wait<0>();
    const uint32_t last_row = ring_g[((nrounds - 1) % STAGES) * STAGEW + (K - 1) * ROWW] & a.kmask[0];
    __syncwarp();
    // chunk epilogue: the still-open row goes to the first (seg == 0) or last partial-row entry
    float* const s_last = reinterpret_cast<float*>(ring);               // [NPW][R], aliases the ring
    {
        float* dst = (seg == 0) ? &s_first[warp][g][sub * V] : s_last + g * R + sub * V;
        vstore<V>(dst, t[0]);
        if (sub == 0) {
            s_erow[warp][2 * g + (seg == 0 ? 0 : 1)] = (int)last_row;
            if (seg == 0) s_erow[warp][2 * g + 1] = -1;
        }
    }
    if (lane == 0) { s_wrow[2 * warp] = -1; s_wrow[2 * warp + 1] = -1; }
    __syncwarp();

    // level 1: merge this warp's 2*NPW partial rows; interior rows are complete -> plain stores
    {
        const float* firsts = &s_first[warp][0][0];
        constexpr int CPL = (R + 31) / 32;
        float acc[CPL];
#pragma unroll
        for (int q = 0; q < CPL; ++q) acc[q] = 0.f;
        int cur_row = -1, run = 0;
        auto emit = [&](int row, bool is_last) {
            float* dst;
            if (run == 0) { dst = &s_wvec[2 * warp][0]; if (lane == 0) s_wrow[2 * warp] = row; }
            else if (is_last) { dst = &s_wvec[2 * warp + 1][0]; if (lane == 0) s_wrow[2 * warp + 1] = row; }
            else dst = a.out + (size_t)row * R;
#pragma unroll
            for (int q = 0; q < CPL; ++q) {
                const int col = lane + 32 * q;
                if (col < R) dst[col] = acc[q];
            }
            ++run;
        };
        for (int e = 0; e < 2 * NPW; ++e) {
            const int r = s_erow[warp][e];
            if (r < 0) continue;
            if (r != cur_row) {
                if (cur_row >= 0) emit(cur_row, false);
                cur_row = r;
#pragma unroll
                for (int q = 0; q < CPL; ++q) acc[q] = 0.f;
            }
            const float* v = (e & 1) ? s_last + (e >> 1) * R : firsts + (e >> 1) * R;
#pragma unroll
            for (int q = 0; q < CPL; ++q) {
                const int col = lane + 32 * q;
                if (col < R) acc[q] += v[col];
            }
        }
        if (cur_row >= 0) emit(cur_row, true);
    }
    __syncthreads();

    // level 2: merge the warps' partial rows; rows shared with a neighbouring shard go to the carry buffer
    if (warp == 0) {
        auto key0_at = [&](int64_t pos) { return __ldg(a.rec + (size_t)pos * RECW) & a.kmask[0]; };   // k_0 sits in word 0
        const uint32_t first_row = key0_at(s_begin);
        const uint32_t end_row = key0_at(s_end - 1);
        const bool head_shared = s_begin > 0 && key0_at(s_begin - 1) == first_row;
        const bool tail_shared = s_end < a.nnz && key0_at(s_end) == end_row;
        constexpr int CPL = (R + 31) / 32;
        merge_runs<R>(s_wrow, &s_wvec[0][0], 2 * WARPS, lane, [&](int row, const float* acc, bool, bool) {
            float* dst;
            if ((uint32_t)row == first_row && head_shared) dst = a.carry + (size_t)(2 * shard) * R;
            else if ((uint32_t)row == end_row && tail_shared) dst = a.carry + (size_t)(2 * shard + 1) * R;
            else dst = a.out + (size_t)row * R;
#pragma unroll
            for (int q = 0; q < CPL; ++q) {
                const int col = lane + 32 * q;
                if (col < R) dst[col] = acc[q];
            }
        });
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
static mttkrp_status_t launch_nr(mttkrp_handle_s* h, int d, const float* const* factors, float* out, cudaStream_t st) {
    const ModeMeta& mm = h->mode[d];
    if (mm.n_empty > 0) {
        const int64_t groups = mm.n_empty;
        const int64_t threads = groups * (R / 4);
        const unsigned grid = (unsigned)std::min<int64_t>((threads + 255) / 256, (int64_t)h->num_sms * 16);
        TimedLaunch tl(h->timing, kClsZero, st);
        k_zero_rows<R><<<grid, 256, 0, st>>>(mm.empty_rows, mm.n_empty, out);
    }
    if (h->num_shards > 0) {
        KernelArgs<N> a;
        a.rec = h->rec_cur;
        a.nnz = h->num_shards * (int64_t)h->shard_nnz;
        a.shard_nnz = h->shard_nnz;
        a.fac[0] = nullptr;
        for (int l = 1; l < N; ++l) a.fac[l] = factors[mm.order[l]];
        a.out = out;
        a.carry = h->carry;
        // Factor matrices that overflow L2 (126 MB) turn gather misses into random HBM reads: use the
        // variant with the deeper look-ahead (measured on configs[2]: 2.96 vs 3.19 ms per mode).
        int64_t fac_bytes = 0;
        for (int l = 1; l < N; ++l) fac_bytes += h->dims[mm.order[l]] * (int64_t)R * 4;
        const bool deep = N <= 3 && (h->force_deep >= 0 ? h->force_deep == 1 : fac_bytes > (96ll << 20));
        for (int l = 0; l < N; ++l) { a.kmask[l] = 0xffffffffu; a.koff[l] = 0; }
        if (h->packed)
            for (int l = 0; l < N; ++l) { a.kmask[l] = pk_mask(mm.pk.bits[l]); a.koff[l] = mm.pk.off[l]; }
        auto launch = [&](auto deep_tag, auto packed_tag) -> mttkrp_status_t {
            constexpr bool DEEP = decltype(deep_tag)::value;
            constexpr bool PACKED = decltype(packed_tag)::value;
            constexpr int smem = Geo<N, R, DEEP, PACKED>::SMEM_BYTES;
            if constexpr (smem > 48 * 1024)               // per device, so not cached in a static
                MK_CUDA(cudaFuncSetAttribute(k_mttkrp<N, R, DEEP, PACKED>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            TimedLaunch tl(h->timing, kClsMttkrp, st);
            k_mttkrp<N, R, DEEP, PACKED><<<(unsigned)h->num_shards, kBlockThreads, smem, st>>>(a);
            return MTTKRP_OK;
        };
        if constexpr (N <= 3) {
            if (deep) MK_TRY(launch(std::true_type{}, std::false_type{}));
            else MK_TRY(launch(std::false_type{}, std::false_type{}));
        } else {
            if (h->packed) MK_TRY(launch(std::false_type{}, std::true_type{}));
            else MK_TRY(launch(std::false_type{}, std::false_type{}));
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
static mttkrp_status_t launch_n(mttkrp_handle_s* h, int d, const float* const* factors, int R, float* out, cudaStream_t st) {
    switch (R) {
        case 8: return launch_nr<N, 8>(h, d, factors, out, st);
        case 16: return launch_nr<N, 16>(h, d, factors, out, st);
        case 32: return launch_nr<N, 32>(h, d, factors, out, st);
        case 64: return launch_nr<N, 64>(h, d, factors, out, st);
    }
    set_error("unsupported rank %d (8, 16, 32, 64)", R);
    return MTTKRP_EUNSUPPORTED;
}

// The resident copy must already be in layout d (api.cu runs the remap passes first).
mttkrp_status_t launch_mttkrp(mttkrp_handle_s* h, int d, const float* const* factors, int R, float* out, cudaStream_t st) {
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
