// spMTTKRP for one mode on the mode-d layout (Alg. 2 "Elementwise Computation", PAPER.md:197-217;
// Alg. 4 thread-block mapping, as function only; the mapping here is this
// library's own, made for sm_100a).
//
// Layout: records sorted by the key tuple (k_0 = i_d, k_1, ..., k_{N-1}); record = N uint32 keys in
// that order + fp32 value, or (N >= 4, PACKED) 16 bytes with the keys bit-packed (common.cuh PackDesc).
// The record carries the run-end flags that the format builder and the remap pass derived from the
// sorted order (bit 31 of key words 0..N-2 / top bits of w1, common.cuh), so it is self-contained: the
// hot loop has no look-ahead compare, and the last key word is flag-free (one multiply-add -> address).
// A thread block owns one shard = shard_nnz consecutive records (equal-nnz shards).  Inside the
// block a GROUP of R/4 lanes (4 rank columns per lane, one 128-bit LDG per factor row per lane:
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
// The kernel is bound by the L1 data pipe (one 128-byte wavefront per clock per SM; every gathered row
// is one) and, next, by instruction issue, so the loop body is kept to what the data needs
// (profiles/r2_sass_hot_loop.md): one LDS.128 per record, one multiply-add per row address, sign tests
// for the flags, and a warp-uniform branch (one vote) around the rare output-row end.
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
    int32_t koff[N];         // unpacked: kmask[l] = kKeyMask
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

struct Vec {                 // 4 rank columns of one lane, as fp32 pairs
    float2 p[2];
};
__device__ __forceinline__ Vec vzero() {
    Vec r;
    r.p[0] = make_float2(0.f, 0.f);
    r.p[1] = make_float2(0.f, 0.f);
    return r;
}

// The record stream is read with an L2 evict-first policy, so that it does not push the factor rows (the data that is
// re-used) out of L2 (measured: -2 % on configs[1], -1 % on configs[2]; an evict-last hint on the factor rows
// themselves was 10 % slower).
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// One lane's 4 columns of a factor row (read-only path, 128-bit load).  `base` = this lane's slot in row 0 of
// the factor matrix (float4 units), `key` = row index, LPN = lanes per row: the address is one 32x32->64
// multiply-add on a per-lane base.  Needs dims[m] < 2^28 (api.cu check_shape).
// (Per-row L2 eviction policies and per-level L1 eviction priorities on these gathers were measured in rounds 1-2 and
// all lost to the plain read-only load; the numbers are in DESIGN.md Sec. 6, the switches are gone.)
template <int LPN>
__device__ __forceinline__ Vec ld_row(const float4* __restrict__ base, uint32_t key) {
    const float4 v = __ldg(base + (size_t)key * LPN);
    Vec r;
    r.p[0] = make_float2(v.x, v.y);
    r.p[1] = make_float2(v.z, v.w);
    return r;
}
// Same for a key word that still carries its run-end flag in bit 31 (fiber levels): the element offset
// (word * LPN + sub) is formed in 32 bits - the shift drops the flag - and scaled by one multiply-add on the
// uniform base, so no mask and no per-lane pointer registers are needed.
template <int LPN>
__device__ __forceinline__ Vec ld_row_flagged(const float* __restrict__ base, uint32_t word, uint32_t sub) {
    constexpr int SH = LPN == 16 ? 4 : (LPN == 8 ? 3 : (LPN == 4 ? 2 : 1));
    const uint32_t off = ((SH >= 2 ? word : (word & kKeyMask)) << SH) + sub;      // the shift drops bits 30 / 31 (flag, cold mark)
    const float4 v = __ldg(reinterpret_cast<const float4*>(base) + off);
    Vec r;
    r.p[0] = make_float2(v.x, v.y);
    r.p[1] = make_float2(v.z, v.w);
    return r;
}
// acc += a * b (elementwise), acc += s * b
__device__ __forceinline__ void vfma(Vec& acc, const Vec& a, const Vec& b) {
    acc.p[0] = ffma2(a.p[0], b.p[0], acc.p[0]);
    acc.p[1] = ffma2(a.p[1], b.p[1], acc.p[1]);
}
__device__ __forceinline__ void vfmas(Vec& acc, float s, const Vec& b) {
    const float2 ss = splat2(s);
    acc.p[0] = ffma2(ss, b.p[0], acc.p[0]);
    acc.p[1] = ffma2(ss, b.p[1], acc.p[1]);
}
__device__ __forceinline__ void vstore(float* dst, const Vec& v) {
    *reinterpret_cast<float4*>(dst) = make_float4(v.p[0].x, v.p[0].y, v.p[1].x, v.p[1].y);
}

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, uint64_t policy) {
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "l"(policy) : "memory");
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
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
// Requests the line of a factor row into L2 (SASS CCTL.E.PF2: no register, no scoreboard).
// One request per row (requesting both 64-byte halves measured slower).
__device__ __forceinline__ void prefetch_l2(const float4* row) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(row));
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

// ---- compile-time geometry ---------------------------------------------------------------------
constexpr int kLookAhead = 2;        // gather look-ahead of the default variant, in steps
constexpr int kLookAheadDeep = 4;    // ... of the DEEP variant
constexpr int kRingStages = 3;       // record ring: round r computing, r+1 landed, the rest in flight
template <int N, int R, bool DEEP, bool PACKED>
struct Geo {
    static constexpr int V = 4;                          // rank columns per lane
    static constexpr int LPN = R / V;                    // lanes per nonzero (group size)
    static constexpr int NPW = 32 / LPN;                 // groups per warp
    static constexpr int WARPS = kBlockThreads / 32;
    static constexpr int G = WARPS * NPW;                // groups per block
    static constexpr int RECW = PACKED ? 4 : N + 1;      // record words
    static constexpr int SLOTW = (RECW + 3) / 4 * 4;     // ring slot words (16-byte multiple)
    static constexpr int K = (NPW * SLOTW <= 32) ? 8 : 4;  // records per group per ring stage
    static constexpr int STAGES = kRingStages;           // round r computing, r+1 landed, the rest in flight
    // gather look-ahead, in steps (K % D == 0).  DEEP: twice the look-ahead at fewer blocks per SM, for
    // factor matrices that do not fit L2 (every gather that misses is a random HBM access).
    static constexpr int D0 = (DEEP && N <= 3) ? kLookAheadDeep : kLookAhead;
    static constexpr int D = (D0 < K) ? D0 : K / 2;
    static constexpr int RING_WORDS = STAGES * K * NPW * SLOTW;        // per warp
    static constexpr int ENT_WORDS = 2 * NPW * R;                       // per warp: first/last partial rows
    static constexpr int WARP_WORDS = RING_WORDS > ENT_WORDS ? RING_WORDS : ENT_WORDS;
    static constexpr int NL = N - 1;                     // accumulator levels t[0..NL-1]
    // resident blocks per SM the register allocation must allow: no instantiation spills, and on B200 (configs[1],
    // configs[2]) occupancy beat deeper look-ahead
    static constexpr int MINB = N <= 3 ? (DEEP ? 3 : 5) : (N == 4 ? (PACKED ? 4 : 3) : (N == 5 ? 3 : 2));
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

// One piece of the mode-d layout, processed by one thread block: `count` records starting at position s_begin.
//   BINS == false (default policy, equal-nnz shards): count == shard_nnz, `fast` is true; rows shared with the
//     neighbouring shards leave their partials in the carry buffer (k_fixup sums them).
//   BINS == true (the paper's Alg. 1 policy: whole output rows dealt to kappa partitions, one
//     thread block per partition, k_mttkrp_bins): the block calls this for the consecutive pieces of its
//     partition [.., seg_end); a row that continues into the next piece is carried in shared memory by the same
//     block, so there is neither a carry buffer nor a fix-up pass.  The ragged last piece (count < shard_nnz,
//     `fast` false) is walked with a plain loop.
//   FUSE == true (MTTKRP_FUSE=1, 16-byte records): the block also executes Alg. 3 for its records, as the paper's
//     kernel does (Alg. 4 lines 15-19): T_out[remap id for mode (d+1) mod N] = record.
template <int N, int R, bool DEEP, bool PACKED, bool BINS, bool FUSE>
__device__ __forceinline__ void shard_body(const KernelArgs<N>& a, const int64_t s_begin, const int count, const bool fast,
                                           const int64_t seg_end, const FuseArgs& fa) {
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
    float* const s_open = reinterpret_cast<float*>(&s_wrow[2 * WARPS]);  // BINS: the row carried into the next piece
    int* const s_open_row = reinterpret_cast<int*>(s_open + R);

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane / LPN, sub = lane % LPN;
    // Default policy: the record array is padded to a whole number of shards (value 0, keys of the last nonzero),
    // so every chunk holds exactly C records and the fast loop needs no bounds checks.
    const int64_t s_end = s_begin + count;
    const int C = fast ? a.shard_nnz / G : (count + G - 1) / G;          // records per group; fast: a multiple of K, > D
    const int nrounds = C / K;
    const int64_t cb = s_begin + min((int64_t)(warp * NPW + g) * C, (int64_t)count);         // this group's first position
    const int64_t ce = s_begin + min((int64_t)(warp * NPW + g + 1) * C, (int64_t)count);     // one past its last
    const uint32_t* const grec = a.rec + (size_t)cb * RECW;

    uint32_t* const ring = &s_warp[warp][0];
    const uint32_t* const ring_g = ring + g * SLOTW;      // this group's column of the ring
    uint32_t ring_gs = (uint32_t)__cvta_generic_to_shared(ring_g);
    asm volatile("mov.u32 %0, %0;" : "+r"(ring_gs));     // opaque: kept in a register instead of being re-derived from %tid every round

    // per-lane bases of the factor rows: row r of level l = fb[l] + r * LPN (float4 units)
    const float4* fb[N];
#pragma unroll
    for (int l = 1; l < N; ++l) fb[l] = reinterpret_cast<const float4*>(a.fac[l]) + sub;
    const float* fiber_base = NL >= 2 ? a.fac[NL >= 2 ? NL - 1 : 1] : nullptr;

    // ---- record ring fill ---------------------------------------------------------------------------------
    const uint64_t rec_policy = l2_policy_evict_first();
    // 16-byte records: piece p of the round = record p of the group, copied by lane p % LPN; the source
    // pointer just advances by one round per call.
    const uint32_t* fill_src = grec + (size_t)sub * RECW;
    uint32_t fill_dst = ring_gs + 4u * (uint32_t)(sub * ROWW);           // ring slot of record `sub` in stage 0
    asm volatile("mov.u32 %0, %0;" : "+r"(fill_dst));
    int fill_round = 0, fill_stage = 0;
    auto issue_round = [&]() {
        if (fill_round < nrounds) {
            const uint32_t dst = ring_gs + 4u * (uint32_t)(fill_stage * STAGEW);
            if constexpr (PPR == 1) {
                const uint32_t dl = fill_dst + 4u * (uint32_t)(fill_stage * STAGEW);
#pragma unroll
                for (int i = 0; i < NPIECE; ++i) {
                    const int p = sub + i * LPN;
                    if (NPIECE * LPN == K || p < K) cp_async16(dl + 4u * (uint32_t)(i * LPN * ROWW), fill_src + (size_t)i * LPN * RECW, rec_policy);
                }
                fill_src += K * RECW;
            } else {
                const uint32_t* src = grec + (size_t)fill_round * (K * RECW);
#pragma unroll
                for (int i = 0; i < NPIECE; ++i) {
                    const int p = sub + i * LPN;
                    if (p < K * PPR) {
                        const int jj = p / PPR, q = p % PPR;
                        const uint32_t d2 = dst + 4u * (uint32_t)(jj * ROWW + q * PW);
                        if constexpr (PW == 2) cp_async8(d2, src + jj * RECW + q * PW);
                        else cp_async4(d2, src + jj * RECW + q * PW);
                    }
                }
            }
        }
        ++fill_round;
        fill_stage = (fill_stage + 1 == STAGES) ? 0 : fill_stage + 1;
        cp_async_commit();
    };

    Vec t[NL];                                            // t[0] = output row accumulator
#pragma unroll
    for (int l = 0; l < NL; ++l) t[l] = vzero();
    bool first_done = false;                              // the chunk's first output-row segment has been emitted
    // Emits the output row that ends at the record whose word 0 is `w0` (run-end flag masked off by the caller's test).
    auto emit_row = [&](uint32_t row) {
        if (!first_done) {
            vstore(&s_first[warp][g][sub * V], t[0]);
            if (sub == 0) s_erow[warp][2 * g] = (int)row;
        } else {
            vstore(a.out + (size_t)row * R + sub * V, t[0]);
        }
        first_done = true;
        t[0] = vzero();
    };
    constexpr bool BATCH = DEEP && N <= 3 && K == 8 && !PACKED;
    uint32_t lw[SLOTW];                                   // the chunk's last record
    bool has = true;                                      // the group has at least one record (always, on the fast path)
    if (!BINS || fast) {
        if constexpr (BATCH) {
            // ---- batch variant (N <= 3) -------------------------------------------------------------------------
            // ptxas tracks every factor-row LDG of this loop on ONE scoreboard, so any wait drains all gathers in
            // flight: a software pipeline degenerates into "issue, wait for everything, compute"
            // (profiles/r2_sass_hot_loop.md).  This variant makes that structure explicit and deep: the records of B = 4
            // steps are read with back-to-back LDS.128, their B last-level rows and up to B fiber rows are requested
            // together (up to 8 independent 128-bit gathers per lane in flight), then the B steps are computed.  Costs
            // 80 registers (3 blocks per SM); one vote per batch replaces the per-step output-row-end test.
            constexpr int B = 4;                                  // (2 and 8 measured slower on configs[2])
            static_assert(K % B == 0, "batch");
            Vec al[B], rb[B];
            float val[B];
            bool e1[B];
            uint32_t anyend = 0;                              // OR of the batch's word 0: sign set = some output row ends in it
            auto batch_prefetch = [&](uint32_t base) {                     // `base` = ring byte address of the batch's first record
                uint4 q[B];
#pragma unroll
                for (int s = 0; s < B; ++s) q[s] = lds128(base + 4u * (uint32_t)(s * ROWW));
                anyend = 0;
#pragma unroll
                for (int s = 0; s < B; ++s) {
                    if constexpr (N == 3) {
                        al[s] = ld_row<LPN>(fb[2], q[s].z);
                        e1[s] = (int32_t)q[s].y < 0;
                        if (e1[s]) rb[s] = ld_row_flagged<LPN>(fiber_base, q[s].y, sub);
                        val[s] = __uint_as_float(q[s].w);
                    } else {
                        al[s] = ld_row<LPN>(fb[1], q[s].y);
                        e1[s] = false;
                        val[s] = __uint_as_float(q[s].z);
                    }
                    anyend |= q[s].x;
                }
            };
            auto batch_compute = [&](uint32_t base) {
                if (!__any_sync(0xffffffffu, (int32_t)anyend < 0)) {      // common: no output row ends in this batch
#pragma unroll
                    for (int s = 0; s < B; ++s) {
                        vfmas(t[NL - 1], val[s], al[s]);
                        if constexpr (N == 3) {
                            if (e1[s]) { vfma(t[0], rb[s], t[1]); t[1] = vzero(); }
                        }
                    }
                } else {
#pragma unroll
                    for (int s = 0; s < B; ++s) {
                        vfmas(t[NL - 1], val[s], al[s]);
                        if constexpr (N == 3) {
                            if (e1[s]) { vfma(t[0], rb[s], t[1]); t[1] = vzero(); }
                        }
                        const uint32_t w0 = lds32(base + 4u * (uint32_t)(s * ROWW));
                        if ((int32_t)w0 < 0) emit_row(w0 & kKeyMask);
                    }
                }
            };
#pragma unroll
            for (int r = 0; r < AHEAD; ++r) issue_round();
            cp_async_wait<AHEAD - 1>();                       // round 0 has landed
            __syncwarp();
            batch_prefetch(ring_gs);
            int stage = 0;
            for (int r = 0; r < nrounds; ++r) {
                issue_round();                                // round r+AHEAD, reuses the stage of round r-1
                constexpr int PF_DIST = 1;                    // rounds between the L2 prefetch of a cold row and its gather (STAGES >= PF_DIST + 2)
                static_assert(AHEAD >= PF_DIST, "prefetch distance");
                cp_async_wait<AHEAD - PF_DIST>();             // rounds <= r+PF_DIST have landed
                __syncwarp();
                const int nstage = (stage + 1 == STAGES) ? 0 : stage + 1;
                const uint32_t cs = ring_gs + 4u * (uint32_t)(stage * STAGEW);
                const uint32_t ns = ring_gs + 4u * (uint32_t)(nstage * STAGEW);
                const uint32_t ps = ring_gs + 4u * (uint32_t)(((stage + PF_DIST) % STAGES) * STAGEW);
                // Cold rows (common.cuh: outside the K most frequent of their factor matrix, so they almost always miss
                // L2 when the factors overflow it) of the NEXT round are requested into L2 now, one round (~3000 clk)
                // before their gathers; lane p of the group looks at record p of that round.  The batch then waits for
                // L2 hits instead of HBM reads (configs[2]: -7 % per mode).
                if (r + PF_DIST < nrounds) {
#pragma unroll
                    for (int i = 0; i < (K + LPN - 1) / LPN; ++i) {
                        const int pr = sub + i * LPN;
                        if (K % LPN == 0 || pr < K) {
                            const uint4 q = lds128(ps + 4u * (uint32_t)(pr * ROWW));
                            const uint32_t klast = N == 3 ? q.z : q.y;
                            if (q.x & kCold) prefetch_l2(reinterpret_cast<const float4*>(a.fac[N - 1]) + (size_t)klast * LPN);
                            if constexpr (N == 3) {
                                if ((int32_t)q.y < 0 && (q.y & kCold))
                                    prefetch_l2(reinterpret_cast<const float4*>(a.fac[1]) + (size_t)(q.y & kKeyMask) * LPN);
                            }
                        }
                    }
                }
#pragma unroll
                for (int b = 0; b < K / B; ++b) {
                    batch_compute(cs + 4u * (uint32_t)(b * B * ROWW));
                    if (b + 1 < K / B) batch_prefetch(cs + 4u * (uint32_t)((b + 1) * B * ROWW));
                    else if (r + 1 < nrounds) batch_prefetch(ns);
                }
                stage = nstage;
                __syncwarp();                                 // everyone is done with round r's stage
            }
        } else {
            Vec al[D];                                            // last-level rows for the D steps in flight
            Vec rb[NL][D];                                        // rb[l][slot]: row of level l, gathered at the end of its run
            float val[D];
            bool e[NL][D];                                        // e[l][slot]: the run of level l ends at that step

            // Issue the gathers of one step whose record sits at ring byte address `slot`.
            auto prefetch = [&](uint32_t slot, int s) {
                uint32_t w[SLOTW];
#pragma unroll
                for (int i = 0; i < SLOTW / 4; ++i) {
                    const uint4 v = lds128(slot + 16u * i);
                    w[4 * i] = v.x; w[4 * i + 1] = v.y; w[4 * i + 2] = v.z; w[4 * i + 3] = v.w;
                }
                if constexpr (PACKED) {                           // {w0, w1 = flags | keys, w2 = last key, val}
                    al[s] = ld_row<LPN>(fb[N - 1], w[2]);
#pragma unroll
                    for (int l = 0; l < NL; ++l) e[l][s] = (w[1] & (0x80000000u >> l)) != 0;
#pragma unroll
                    for (int l = 1; l < NL; ++l)
                        if (e[l][s]) rb[l][s] = ld_row_flagged<LPN>(a.fac[l], pk_get(w[0], w[1], a.koff[l], a.kmask[l]), sub);
                    val[s] = __uint_as_float(w[3]);
                } else {
                    al[s] = ld_row<LPN>(fb[N - 1], w[N - 1]);
#pragma unroll
                    for (int l = 0; l < NL; ++l) e[l][s] = (int32_t)w[l] < 0;
                    if constexpr (NL >= 2) {
                        if (e[NL - 1][s]) rb[NL - 1][s] = ld_row_flagged<LPN>(fiber_base, w[NL - 1], sub);
                    }
#pragma unroll
                    for (int l = 1; l < NL - 1; ++l)
                        if (e[l][s]) rb[l][s] = ld_row_flagged<LPN>(a.fac[l], w[l], sub);
                    val[s] = __uint_as_float(w[N]);
                }
            };
            // Arithmetic of one step (its record sits at `slot`).
            auto compute = [&](uint32_t slot, int s) {
                vfmas(t[NL - 1], val[s], al[s]);
                if constexpr (NL >= 2) {
                    if (e[NL - 1][s]) {
                        vfma(t[NL - 2], rb[NL - 1][s], t[NL - 1]);
                        t[NL - 1] = vzero();
                    }
                }
                // upper fiber levels: plain predication (a vote + branch per level takes the scheduler's freedom to hoist
                // the gathers: measured 10-28 % slower for N = 4, 5)
#pragma unroll
                for (int l = NL - 2; l >= 1; --l) {
                    if (e[l][s]) {
                        vfma(t[l - 1], rb[l][s], t[l]);
                        t[l] = vzero();
                    }
                }
                if (__any_sync(0xffffffffu, e[0][s])) {           // rare: an output row ends inside the chunk
                    // Every lane reads its group's row id first (a volatile load): the branch above then depends on the
                    // vote alone and stays warp-uniform; only the stores below are per lane.
                    uint32_t row;
                    if constexpr (PACKED) row = pk_get(lds32(slot), lds32(slot + 4), a.koff[0], a.kmask[0]);
                    else row = lds32(slot) & kKeyMask;
                    if (e[0][s]) emit_row(row);
                }
            };

            // Dynamic tensor remapping inside the compute kernel (FUSE): lane p % LPN moves record p of the round.  The
            // remap id and the next layout's flags are fetched at the start of the round, the record is re-read from
            // the ring after the round's arithmetic, re-ordered for the next layout and scattered (Alg. 3).
            uint32_t f_dst[NPIECE], f_fl[NPIECE];
            auto fuse_load = [&](int r) {
#pragma unroll
                for (int i = 0; i < NPIECE; ++i) {
                    const int p = sub + i * LPN;
                    const int64_t pos = cb + (int64_t)r * K + p;
                    f_dst[i] = 0xffffffffu;
                    if (p < K && pos < fa.nnz) { f_dst[i] = __ldg(fa.scat + pos); f_fl[i] = __ldg(fa.sflags + pos); }
                }
            };
            auto fuse_store = [&](uint32_t cs) {
#pragma unroll
                for (int i = 0; i < NPIECE; ++i) {
                    const int p = sub + i * LPN;
                    if (p < K && f_dst[i] != 0xffffffffu) {
                        const uint4 q = lds128(cs + 4u * (uint32_t)(p * ROWW));
                        uint32_t k[N];
                        uint4 o;
                        if constexpr (PACKED) {
#pragma unroll
                            for (int l = 0; l < N; ++l)
                                k[l] = fa.rp.soff[l] < 0 ? (q.z & fa.rp.smask[l]) : pk_get(q.x, q.y, fa.rp.soff[l], fa.rp.smask[l]);
                            o = pk_pack<N>(k, f_fl[i], q.w, fa.dd);
                        } else {
                            const uint32_t f[3] = {q.x & kKeyMask, q.y & kKeyMask, q.z & kKeyMask};
#pragma unroll
                            for (int l = 0; l < 3; ++l) k[l] = fa.fm.src[l] == 0 ? f[0] : (fa.fm.src[l] == 1 ? f[1] : f[2]);
                            apply_run_flags<3>(k, f_fl[i]);
                            o = make_uint4(k[0], k[1], k[2], q.w);
                        }
                        *(reinterpret_cast<uint4*>(fa.out_rec) + f_dst[i]) = o;
                    }
                }
            };

            // ---- prologue: rounds 0..AHEAD-1 in flight, round 0 landed ----------------------------------------
#pragma unroll
            for (int r = 0; r < AHEAD; ++r) issue_round();
            cp_async_wait<AHEAD - 1>();                           // round 0 has landed
            __syncwarp();
#pragma unroll
            for (int i = 0; i < D; ++i) prefetch(ring_gs + 4u * (uint32_t)(i * ROWW), i);
            int stage = 0;                                        // r % STAGES
            for (int r = 0; r < nrounds; ++r) {
                issue_round();                                    // round r+AHEAD, reuses the stage of round r-1
                cp_async_wait<AHEAD - 1>();                       // rounds <= r+1 have landed
                __syncwarp();
                const int nstage = (stage + 1 == STAGES) ? 0 : stage + 1;
                const uint32_t cs = ring_gs + 4u * (uint32_t)(stage * STAGEW);            // this round's stage
                const uint32_t ns = ring_gs + 4u * (uint32_t)(nstage * STAGEW);           // next round's stage
                const bool more = r + 1 < nrounds;
                if constexpr (FUSE) fuse_load(r);
#pragma unroll
                for (int i = 0; i < K; ++i) {
                    compute(cs + 4u * (uint32_t)(i * ROWW), i % D);
                    if (i + D < K) prefetch(cs + 4u * (uint32_t)((i + D) * ROWW), i % D);
                    else if (more) prefetch(ns + 4u * (uint32_t)((i + D - K) * ROWW), i % D);
                }
                if constexpr (FUSE) fuse_store(cs);
                stage = nstage;
                __syncwarp();                                     // everyone is done with round r's stage
            }
        }
        cp_async_wait<0>();
        __syncwarp();
        const uint32_t* const last_rec = ring_g + ((nrounds - 1) % STAGES) * STAGEW + (K - 1) * ROWW;
#pragma unroll
        for (int i = 0; i < SLOTW; ++i) lw[i] = last_rec[i];
    } else {
        // ragged piece (BINS only): one record at a time straight from global memory, gathers not overlapped
        has = ce > cb;
        for (int64_t pos = cb; pos < ce; ++pos) {
            const uint32_t* rp = a.rec + (size_t)pos * RECW;
#pragma unroll
            for (int i = 0; i < RECW; ++i) lw[i] = __ldg(rp + i);
            uint32_t key[N];
            bool en[NL];
            float v;
            if constexpr (PACKED) {
#pragma unroll
                for (int l = 0; l < NL; ++l) { key[l] = pk_get(lw[0], lw[1], a.koff[l], a.kmask[l]); en[l] = (lw[1] & (0x80000000u >> l)) != 0; }
                key[N - 1] = lw[2];
                v = __uint_as_float(lw[3]);
            } else {
#pragma unroll
                for (int l = 0; l < NL; ++l) { key[l] = lw[l] & kKeyMask; en[l] = (int32_t)lw[l] < 0; }
                key[N - 1] = lw[N - 1];
                v = __uint_as_float(lw[N]);
            }
            vfmas(t[NL - 1], v, ld_row<LPN>(fb[N - 1], key[N - 1]));
#pragma unroll
            for (int l = NL - 1; l >= 1; --l) {
                if (en[l]) { vfma(t[l - 1], ld_row<LPN>(fb[l], key[l]), t[l]); t[l] = vzero(); }
            }
            if (en[0]) emit_row(key[0]);
        }
    }
    // ---- chunk epilogue -----------------------------------------------------------------------------------
    // The chunk's last record leaves its inner runs open unless they end there: fold them now (the level's
    // row is the last record's key), so that t[0] holds everything the chunk contributes to its last row.
    if (has) {
#pragma unroll
        for (int l = NL - 1; l >= 1; --l) {
            bool ended;
            uint32_t key;
            if constexpr (PACKED) { ended = (lw[1] & (0x80000000u >> l)) != 0; key = pk_get(lw[0], lw[1], a.koff[l], a.kmask[l]); }
            else { ended = (int32_t)lw[l] < 0; key = lw[l] & kKeyMask; }
            if (!ended) {
                const Vec row = ld_row<LPN>(fb[l], key);
                vfma(t[l - 1], row, t[l]);
                t[l] = vzero();
            }
        }
    }
    bool last_open = false;                               // the chunk's last output row continues past the chunk
    uint32_t last_row = 0;
    if (has) {
        if constexpr (PACKED) { last_open = (lw[1] & 0x80000000u) == 0; last_row = pk_get(lw[0], lw[1], a.koff[0], a.kmask[0]); }
        else { last_open = (int32_t)lw[0] >= 0; last_row = lw[0] & kKeyMask; }
    }
    __syncwarp();
    // The still-open row goes to the first (nothing emitted yet) or last partial-row entry; a row that ended
    // exactly at the chunk's last record was already emitted by the loop.
    float* const s_last = reinterpret_cast<float*>(ring);               // [NPW][R], aliases the ring
    if (last_open) {
        float* dst = !first_done ? &s_first[warp][g][sub * V] : s_last + g * R + sub * V;
        vstore(dst, t[0]);
    }
    if (sub == 0) {
        if (!has) {
            s_erow[warp][2 * g] = -1;                     // ragged piece: this group got no record
            s_erow[warp][2 * g + 1] = -1;
        } else if (last_open) {
            s_erow[warp][2 * g + (first_done ? 1 : 0)] = (int)last_row;
            if (!first_done) s_erow[warp][2 * g + 1] = -1;
        } else {
            s_erow[warp][2 * g + 1] = -1;                 // first_done here: entry 0 was written by the loop
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
        for (int ee = 0; ee < 2 * NPW; ++ee) {
            const int r = s_erow[warp][ee];
            if (r < 0) continue;
            if (r != cur_row) {
                if (cur_row >= 0) emit(cur_row, false);
                cur_row = r;
#pragma unroll
                for (int q = 0; q < CPL; ++q) acc[q] = 0.f;
            }
            const float* v = (ee & 1) ? s_last + (ee >> 1) * R : firsts + (ee >> 1) * R;
#pragma unroll
            for (int q = 0; q < CPL; ++q) {
                const int col = lane + 32 * q;
                if (col < R) acc[q] += v[col];
            }
        }
        if (cur_row >= 0) emit(cur_row, true);
    }
    __syncthreads();

    // level 2: merge the warps' partial rows
    if (warp == 0) {
        auto key0_at = [&](int64_t pos) {
            const uint32_t* p = a.rec + (size_t)pos * RECW;
            if constexpr (PACKED) return pk_get(__ldg(p), __ldg(p + 1), a.koff[0], a.kmask[0]);
            else return __ldg(p) & kKeyMask;                            // k_0 sits in word 0
        };
        constexpr int CPL = (R + 31) / 32;
        if constexpr (!BINS) {
            // rows shared with a neighbouring shard go to the carry buffer (k_fixup sums them in fixed order)
            const int64_t shard = s_begin / a.shard_nnz;
            const uint32_t first_row = key0_at(s_begin);
            const uint32_t end_row = key0_at(s_end - 1);
            const bool head_shared = s_begin > 0 && key0_at(s_begin - 1) == first_row;
            const bool tail_shared = s_end < a.nnz && key0_at(s_end) == end_row;
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
        } else {
            // Alg. 1 policy: the whole partition belongs to this block, so a row that continues into the block's
            // next piece is carried in shared memory (s_open) and stored once, when it ends.
            const bool more = s_end < seg_end;
            const uint32_t next_row = more ? key0_at(s_end) : 0u;
            const int open_row = *s_open_row;
            __syncwarp();
            merge_runs<R>(s_wrow, &s_wvec[0][0], 2 * WARPS, lane, [&](int row, const float* acc, bool, bool is_last) {
                const bool cont_prev = row == open_row;
                const bool cont_next = is_last && more && (uint32_t)row == next_row;
#pragma unroll
                for (int q = 0; q < CPL; ++q) {
                    const int col = lane + 32 * q;
                    if (col < R) {
                        const float v = acc[q] + (cont_prev ? s_open[col] : 0.f);
                        if (cont_next) s_open[col] = v;
                        else a.out[(size_t)row * R + col] = v;
                    }
                }
                if (lane == 0) {
                    if (cont_next) *s_open_row = row;
                    else if (cont_prev) *s_open_row = -1;
                }
            });
        }
    }
}

// Default policy: one thread block per equal-nnz shard.
template <int N, int R, bool DEEP, bool PACKED>
__global__ void __launch_bounds__(kBlockThreads, Geo<N, R, DEEP, PACKED>::MINB) k_mttkrp(const KernelArgs<N> a) {
    shard_body<N, R, DEEP, PACKED, false, false>(a, (int64_t)blockIdx.x * a.shard_nnz, a.shard_nnz, true, 0, FuseArgs());
}

// Same, with the dynamic tensor remapping of Alg. 3 executed by the same kernel (MTTKRP_FUSE=1; 16-byte records).
template <int N, int R, bool PACKED>
__global__ void __launch_bounds__(kBlockThreads, Geo<N, R, false, PACKED>::MINB) k_mttkrp_fused(const KernelArgs<N> a, const FuseArgs fa) {
    shard_body<N, R, false, PACKED, false, true>(a, (int64_t)blockIdx.x * a.shard_nnz, a.shard_nnz, true, 0, fa);
}

// The paper's Alg. 1 policy (Alg. 4/5: one thread block per partition B_{d,z}): block z walks the
// records [bins[z], bins[z+1]) of the partition-ordered layout in pieces of shard_nnz and owns every output row in it.
template <int N, int R, bool PACKED>
__global__ void __launch_bounds__(kBlockThreads, Geo<N, R, false, PACKED>::MINB) k_mttkrp_bins(const KernelArgs<N> a,
                                                                                               const uint32_t* __restrict__ bins) {
    extern __shared__ uint4 smem_raw[];
    int* const s_open_row = reinterpret_cast<int*>(reinterpret_cast<char*>(smem_raw) + Geo<N, R, false, PACKED>::SMEM_BYTES) + R;
    if (threadIdx.x == 0) *s_open_row = -1;
    __syncthreads();
    const int64_t begin = bins[blockIdx.x], end = bins[blockIdx.x + 1];
    for (int64_t p = begin; p < end; p += a.shard_nnz) {
        const int count = (int)min((int64_t)a.shard_nnz, end - p);
        shard_body<N, R, false, PACKED, true, false>(a, p, count, count == a.shard_nnz, end, FuseArgs());
        __syncthreads();                                  // the next piece reuses the shared-memory areas
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
        // variant with the deeper look-ahead.  MTTKRP_FORCE_DEEP (read at create) pins the choice for tests.
        int64_t fac_bytes = 0;
        for (int l = 1; l < N; ++l) fac_bytes += h->dims[mm.order[l]] * (int64_t)R * 4;
        const bool deep = N <= 3 && (h->force_deep >= 0 ? h->force_deep == 1 : fac_bytes > (96ll << 20));
        for (int l = 0; l < N; ++l) { a.kmask[l] = kKeyMask; a.koff[l] = 0; }
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
        auto launch_bins = [&](auto packed_tag) -> mttkrp_status_t {
            constexpr bool PACKED = decltype(packed_tag)::value;
            constexpr int smem = Geo<N, R, false, PACKED>::SMEM_BYTES + 4 * (R + 4);      // + the carried row
            if constexpr (smem > 48 * 1024)
                MK_CUDA(cudaFuncSetAttribute(k_mttkrp_bins<N, R, PACKED>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            TimedLaunch tl(h->timing, kClsMttkrp, st);
            k_mttkrp_bins<N, R, PACKED><<<(unsigned)h->kappa, kBlockThreads, smem, st>>>(a, mm.bins);
            return MTTKRP_OK;
        };
        auto launch_fused = [&](auto packed_tag) -> mttkrp_status_t {
            constexpr bool PACKED = decltype(packed_tag)::value;
            constexpr int smem = Geo<N, R, false, PACKED>::SMEM_BYTES;
            FuseArgs fa;
            const int to = (d + 1) % N;
            fa.out_rec = h->rec_alt;
            fa.scat = mm.scat;
            fa.sflags = mm.sflags;
            fa.nnz = h->nnz;
            remap_fields(h, d, to, &fa.fm, &fa.rp);
            fa.dd = h->mode[to].pk;
            if constexpr (smem > 48 * 1024)
                MK_CUDA(cudaFuncSetAttribute(k_mttkrp_fused<N, R, PACKED>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            TimedLaunch tl(h->timing, kClsMttkrp, st);
            k_mttkrp_fused<N, R, PACKED><<<(unsigned)h->num_shards, kBlockThreads, smem, st>>>(a, fa);
            return MTTKRP_OK;
        };
        if (h->fuse) {                                    // remap inside the compute kernel (Alg. 4 lines 15-19)
            if constexpr (N == 3) MK_TRY(launch_fused(std::false_type{}));
            else if constexpr (N >= 4) { if (h->packed) MK_TRY(launch_fused(std::true_type{})); }
        } else if (h->policy == 1) {                      // the paper's Alg. 1 policy: one block per partition, no fix-up
            if (h->packed) { if constexpr (N >= 4) MK_TRY(launch_bins(std::true_type{})); }
            else MK_TRY(launch_bins(std::false_type{}));
        } else if constexpr (N <= 3) {
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
#ifndef MK_FAST_BUILD
        case 8: return launch_nr<N, 8>(h, d, factors, out, st);
        case 16: return launch_nr<N, 16>(h, d, factors, out, st);
        case 64: return launch_nr<N, 64>(h, d, factors, out, st);
#endif
        case 32: return launch_nr<N, 32>(h, d, factors, out, st);
    }
    set_error("unsupported rank %d (8, 16, 32, 64)", R);
    return MTTKRP_EUNSUPPORTED;
}

// The resident copy must already be in layout d (api.cu runs the remap passes first).
mttkrp_status_t launch_mttkrp(mttkrp_handle_s* h, int d, const float* const* factors, int R, float* out, cudaStream_t st) {
    switch (h->N) {
#ifndef MK_FAST_BUILD                                    // -DMK_FAST_BUILD: N = 3, R = 32 only (SASS inspection)
        case 2: return launch_n<2>(h, d, factors, R, out, st);
        case 4: return launch_n<4>(h, d, factors, R, out, st);
        case 5: return launch_n<5>(h, d, factors, R, out, st);
        case 6: return launch_n<6>(h, d, factors, R, out, st);
        case 7: return launch_n<7>(h, d, factors, R, out, st);
        case 8: return launch_n<8>(h, d, factors, R, out, st);
#endif
        case 3: return launch_n<3>(h, d, factors, R, out, st);
    }
    set_error("unsupported nmodes %d", h->N);
    return MTTKRP_EUNSUPPORTED;
}

}  // namespace mk
