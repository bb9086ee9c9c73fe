// Microbenchmark behind DESIGN.md Sec. 6 ("gather ceiling"): how fast can an SM gather random 128-byte factor rows?
//   * LDG shapes: 32 lanes x 4 B (one row per instruction), 8 lanes x 16 B (four rows), 4 lanes x 32 B (eight rows),
//     from tables that are L1-, L2- or HBM-resident;
//   * LDS from a shared-memory copy of the table (conflict-free shape: 8 lanes x 16 B per row);
//   * per-row cp.async.bulk (TMA) into a shared-memory ring, consumed with LDS;
//   * remap-style record gathers: out[j] = in[prev[j]] for 16- and 32-byte records, uniformly random and from an
//     L2-sized window.
// Not part of the library.  Build and run (one B200):
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o gather_rate paper_2405_08470_b200/csrc/probes/gather_rate.cu
//   ./gather_rate
// ncu wavefront counts: ROWS=29000 ncu --metrics l1tex__data_pipe_lsu_wavefronts_mem_lgds.sum,l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum -k regex:"^k_gather$" ./gather_rate
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <vector>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n", cudaGetErrorString(e), __LINE__); exit(1);} }while(0)

__device__ __forceinline__ uint32_t hash32(uint32_t x){ x^=x>>16; x*=0x7feb352dU; x^=x>>15; x*=0x846ca68bU; x^=x>>16; return x; }

// SHAPE: lanes per row = 32 (4B/lane), 8 (16B/lane), 4 (32B/lane).  Each group of LPR lanes processes rows idx[g + k*G].
template<int LPR, int U>
__global__ void __launch_bounds__(256) k_gather(const float* __restrict__ tab, const uint32_t* __restrict__ idx, int64_t n_per_group, float* out){
    const int tid = blockIdx.x*blockDim.x + threadIdx.x;
    const int64_t group = tid / LPR; const int sub = tid % LPR;
    const uint32_t* ip = idx + group * n_per_group;
    float acc[8] = {0,0,0,0,0,0,0,0};
    for (int64_t k = 0; k < n_per_group; k += U) {
        uint32_t r[U];
        #pragma unroll
        for (int u=0;u<U;++u) r[u] = __ldcs(ip + k + u);
        #pragma unroll
        for (int u=0;u<U;++u) {
            const float* p = tab + (size_t)r[u]*32;
            if constexpr (LPR==32) { acc[0] += __ldg(p+sub); }
            else if constexpr (LPR==8) { float4 v = __ldg((const float4*)p + sub); acc[0]+=v.x; acc[1]+=v.y; acc[2]+=v.z; acc[3]+=v.w; }
            else { float v0,v1,v2,v3,v4,v5,v6,v7; asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];":"=f"(v0),"=f"(v1),"=f"(v2),"=f"(v3),"=f"(v4),"=f"(v5),"=f"(v6),"=f"(v7):"l"(p+sub*8));
                   acc[0]+=v0;acc[1]+=v1;acc[2]+=v2;acc[3]+=v3;acc[4]+=v4;acc[5]+=v5;acc[6]+=v6;acc[7]+=v7; }
        }
    }
    float s=0; for(int i=0;i<8;++i) s+=acc[i];
    if (s == 123.456f) out[tid] = s;
}

// smem-resident table of TR rows: gather with LDS (4 lanes x 2 LDS.128 per row; 2-way bank conflict)
template<int TR, int U>
__global__ void __launch_bounds__(256) k_gather_smem(const float* __restrict__ tab, const uint32_t* __restrict__ idx, int64_t n_per_group, float* out){
    extern __shared__ float4 sm[];
    for (int i = threadIdx.x; i < TR*8; i += 256) sm[i] = ((const float4*)tab)[i];
    __syncthreads();
    const int tid = blockIdx.x*blockDim.x + threadIdx.x;
    const int64_t group = tid / 4; const int sub = tid % 4;
    const uint32_t* ip = idx + group * n_per_group;
    float acc[8] = {0,0,0,0,0,0,0,0};
    for (int64_t k = 0; k < n_per_group; k += U) {
        uint32_t r[U];
        #pragma unroll
        for (int u=0;u<U;++u) r[u] = __ldcs(ip + k + u) & (TR-1);
        #pragma unroll
        for (int u=0;u<U;++u) {
            float4 a = sm[r[u]*8 + sub*2], b = sm[r[u]*8 + sub*2 + 1];
            acc[0]+=a.x;acc[1]+=a.y;acc[2]+=a.z;acc[3]+=a.w;acc[4]+=b.x;acc[5]+=b.y;acc[6]+=b.z;acc[7]+=b.w;
        }
    }
    float s=0; for(int i=0;i<8;++i) s+=acc[i];
    if (s == 123.456f) out[tid] = s;
}

struct alignas(32) R32 { uint4 a,b; };
// remap-style: out[j] = in[prev[j]] with records of RB bytes

template<typename T>
__global__ void k_gather_rec(const T* __restrict__ in, const uint32_t* __restrict__ prev, T* __restrict__ out, int64_t n){
    int64_t j = (int64_t)blockIdx.x*blockDim.x + threadIdx.x;
    if (j<n) { T v = in[__ldcs(prev+j)]; out[j] = v; }
}

__global__ void k_fill_idx(uint32_t* idx, int64_t n, uint32_t mod, uint32_t seed){
    int64_t j = (int64_t)blockIdx.x*blockDim.x + threadIdx.x;
    if (j<n) idx[j] = (uint32_t)(((uint64_t)hash32((uint32_t)j*2654435761u + seed) * mod) >> 32);
}

template<class F> float timeit(F f, int reps=5){
    cudaEvent_t a,b; cudaEventCreate(&a); cudaEventCreate(&b);
    f(); CK(cudaDeviceSynchronize());
    float best=1e30f;
    for(int i=0;i<reps;++i){ cudaEventRecord(a); f(); cudaEventRecord(b); CK(cudaEventSynchronize(b)); float ms; cudaEventElapsedTime(&ms,a,b); if(ms<best)best=ms; }
    return best;
}


// conflict-free smem shape
template<int TR, int U>
__global__ void __launch_bounds__(256) k_gather_smem8(const float* __restrict__ tab, const uint32_t* __restrict__ idx, int64_t npg, float* out){
    extern __shared__ float4 sm[];
    for (int i = threadIdx.x; i < TR*8; i += 256) sm[i] = ((const float4*)tab)[i];
    __syncthreads();
    const int tid = blockIdx.x*blockDim.x + threadIdx.x;
    const int64_t group = tid / 8; const int sub = tid % 8;
    const uint32_t* ip = idx + group * npg;
    float4 acc = make_float4(0,0,0,0);
    for (int64_t k = 0; k < npg; k += U) {
        uint32_t r[U];
        #pragma unroll
        for (int u=0;u<U;++u) r[u] = __ldcs(ip + k + u) & (TR-1);
        #pragma unroll
        for (int u=0;u<U;++u) { float4 a = sm[r[u]*8 + sub]; acc.x+=a.x;acc.y+=a.y;acc.z+=a.z;acc.w+=a.w; }
    }
    if (acc.x+acc.y+acc.z+acc.w == 123.456f) out[tid] = acc.x;
}


// per-row TMA bulk copies
__device__ __forceinline__ void mbar_init(uint32_t a, int c){ asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;"::"r"(a),"r"(c)); }
__device__ __forceinline__ void mbar_expect(uint32_t a, uint32_t tx){ asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"::"r"(a),"r"(tx):"memory"); }
__device__ __forceinline__ void mbar_wait(uint32_t a, uint32_t ph){
    asm volatile("{\n .reg .pred p;\n W: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @p bra D;\n bra W;\n D:\n}"::"r"(a),"r"(ph):"memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t mbar){
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"::"r"(dst),"l"(src),"r"(bytes),"r"(mbar):"memory");
}
// each warp: ring of STAGES slots of 32 rows x 128 B
template<int STAGES, int WARPS>
__global__ void __launch_bounds__(WARPS*32) k_gather_bulk(const float* __restrict__ tab, const uint32_t* __restrict__ idx, int64_t n_per_warp, float* out){
    extern __shared__ __align__(128) unsigned char smraw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned char* ring = smraw + (size_t)warp * STAGES * 4096;
    uint64_t* bars = (uint64_t*)(smraw + (size_t)WARPS*STAGES*4096) + warp*STAGES;
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(ring);
    const uint32_t bars_s = (uint32_t)__cvta_generic_to_shared(bars);
    if (lane == 0) { for (int s=0;s<STAGES;++s) mbar_init(bars_s + 8*s, 1); }
    asm volatile("fence.mbarrier_init.release.cluster;":::"memory");
    __syncwarp();
    const int64_t gw = (int64_t)blockIdx.x*WARPS + warp;
    const uint32_t* ip = idx + gw * n_per_warp;
    const int64_t nsteps = n_per_warp / 32;
    float4 acc = make_float4(0,0,0,0);
    auto issue=[&](int64_t s){
        const int slot = (int)(s % STAGES);
        if (lane == 0) mbar_expect(bars_s + 8*slot, 4096);
        __syncwarp();
        uint32_t r = __ldcs(ip + s*32 + lane);
        bulk_g2s(ring_s + slot*4096 + lane*128, tab + (size_t)r*32, 128, bars_s + 8*slot);
    };
    for (int s=0;s<STAGES-1 && s<nsteps;++s) issue(s);
    for (int64_t s=0;s<nsteps;++s){
        if (s + STAGES-1 < nsteps) issue(s+STAGES-1);
        const int slot = (int)(s % STAGES);
        mbar_wait(bars_s + 8*slot, (uint32_t)((s/STAGES)&1));
        const float4* rp = (const float4*)(ring + slot*4096);
        #pragma unroll
        for (int q=0;q<8;++q){ float4 a = rp[q*32 + lane]; acc.x+=a.x;acc.y+=a.y;acc.z+=a.z;acc.w+=a.w; }   // 4 rows per LDS.128, conflict-free
        __syncwarp();
    }
    if (acc.x+acc.y+acc.z+acc.w == 123.456f) out[threadIdx.x] = acc.x;
}

int main(){
    const int64_t NIDX = 64<<20;   // 64M row gathers per run
    uint32_t* idx; CK(cudaMalloc(&idx, NIDX*4));
    float* out; CK(cudaMalloc(&out, 1<<24));
    const size_t maxrows = 8u<<20;  // 1 GB table
    float* tab; CK(cudaMalloc(&tab, maxrows*128)); CK(cudaMemset(tab, 0, maxrows*128));
    cudaDeviceProp pr; cudaGetDeviceProperties(&pr,0);
    const double clk = 1.965e9; const int sms = pr.multiProcessorCount;
    printf("device %s SMs %d\n", pr.name, sms);
    const int blocks = sms*8;  // 8 CTAs x 256 thr = 2048 thr/SM
    uint32_t rows_list[] = {256, 1024, 4096, 9000, 29000, 65536, 262144, 1u<<20, 8u<<20};
    for (uint32_t rows : rows_list) { if (getenv("QUICK")) break; if (getenv("ROWS") && (uint32_t)atoi(getenv("ROWS")) != rows) continue;
        k_fill_idx<<<(NIDX+255)/256,256>>>(idx, NIDX, rows, 12345u);
        CK(cudaDeviceSynchronize());
        auto report=[&](const char* name, float ms, int64_t total){ double rps = total/(ms*1e-3); printf("rows=%8u (%8.1f KB) %-14s %7.3f ms  %7.1f Grows/s  %6.3f rows/clk/SM  %7.1f GB/s\n", rows, rows*128/1024.0, name, ms, rps/1e9, rps/clk/sms, rps*128/1e9); };
        { const int64_t groups = (int64_t)blocks*256/32; const int64_t npg = NIDX/groups/8*8; float ms = timeit([&]{ k_gather<32,8><<<blocks,256>>>(tab, idx, npg, out); }); report("32x4B U8", ms, npg*groups); }
        { const int64_t groups = (int64_t)blocks*256/8; const int64_t npg = NIDX/groups/8*8; float ms = timeit([&]{ k_gather<8,8><<<blocks,256>>>(tab, idx, npg, out); }); report("8x16B U8", ms, npg*groups); }
        { const int64_t groups = (int64_t)blocks*256/4; const int64_t npg = NIDX/groups/8*8; float ms = timeit([&]{ k_gather<4,4><<<blocks,256>>>(tab, idx, npg, out); }); report("4x32B U4", ms, npg*groups); }
        { const int64_t groups = (int64_t)blocks*256/4; const int64_t npg = NIDX/groups/8*8; float ms = timeit([&]{ k_gather<4,8><<<blocks,256>>>(tab, idx, npg, out); }); report("4x32B U8", ms, npg*groups); }
    }
    if (!getenv("QUICK")) {   // smem gathers
        k_fill_idx<<<(NIDX+255)/256,256>>>(idx, NIDX, 1u<<20, 777u);
        CK(cudaFuncSetAttribute(k_gather_smem<1024,8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 1024*128));
        const int b2 = sms; const int64_t groups=(int64_t)b2*256/4; const int64_t npg = NIDX/groups/8*8;
        float ms = timeit([&]{ k_gather_smem<1024,8><<<b2,256,1024*128>>>(tab, idx, npg, out); });
        double rps = npg*groups/(ms*1e-3); printf("smem 1024 rows, 1 CTA/SM 256thr: %.3f ms %.1f Grows/s %.3f rows/clk/SM\n", ms, rps/1e9, rps/clk/sms);
        CK(cudaFuncSetAttribute(k_gather_smem<512,8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 512*128));
        const int b3 = sms*3; const int64_t groups3=(int64_t)b3*256/4; const int64_t npg3 = NIDX/groups3/8*8;
        ms = timeit([&]{ k_gather_smem<512,8><<<b3,256,512*128>>>(tab, idx, npg3, out); });
        rps = npg3*groups3/(ms*1e-3); printf("smem 512 rows, 3 CTA/SM 256thr: %.3f ms %.1f Grows/s %.3f rows/clk/SM\n", ms, rps/1e9, rps/clk/sms);
    }
    if (!getenv("QUICK")) {   // conflict-free LDS shape and per-row TMA bulk copies (table contents do not matter)
        k_fill_idx<<<(NIDX+255)/256,256>>>(idx, NIDX, 29000u, 4711u); CK(cudaDeviceSynchronize());
        auto report=[&](const char* name, float ms, int64_t total){ double rps = total/(ms*1e-3); printf("%-34s %7.3f ms  %7.1f Grows/s  %6.3f rows/clk/SM\n", name, ms, rps/1e9, rps/clk/sms); fflush(stdout); };
        { CK(cudaFuncSetAttribute(k_gather_smem8<512,8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 512*128));
          const int blocks=sms*3; const int64_t groups=(int64_t)blocks*256/8; const int64_t npg=NIDX/groups/8*8; float ms=timeit([&]{k_gather_smem8<512,8><<<blocks,256,512*128>>>(tab,idx,npg,out);}); report("LDS 8x16B smem 512 rows, 3 CTA/SM",ms,npg*groups); }
        { constexpr int ST=4, W=8; const int smem = W*ST*4096 + W*ST*8; CK(cudaFuncSetAttribute(k_gather_bulk<ST,W>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
          const int blocks=sms; const int64_t warps=(int64_t)blocks*W; const int64_t npw=NIDX/warps/32*32; float ms=timeit([&]{k_gather_bulk<ST,W><<<blocks,W*32,smem>>>(tab,idx,npw,out);}); report("cp.async.bulk 128 B, 8 warps/SM",ms,npw*warps); }
        { constexpr int ST=3, W=4; const int smem = W*ST*4096 + W*ST*8; CK(cudaFuncSetAttribute(k_gather_bulk<ST,W>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
          const int blocks=sms*4; const int64_t warps=(int64_t)blocks*W; const int64_t npw=NIDX/warps/32*32; float ms=timeit([&]{k_gather_bulk<ST,W><<<blocks,W*32,smem>>>(tab,idx,npw,out);}); report("cp.async.bulk 128 B, 16 warps/SM",ms,npw*warps); }
    }
    {   // remap-style record gather: n records, random permutation-ish source
        const int64_t n = 32<<20;
        if (getenv("GRAN")) { CK(cudaDeviceSetLimit(cudaLimitMaxL2FetchGranularity, atoi(getenv("GRAN")))); } size_t gr=0; cudaDeviceGetLimit(&gr, cudaLimitMaxL2FetchGranularity); printf("L2 fetch granularity %zu\n", gr);
        k_fill_idx<<<(n+255)/256,256>>>(idx, n, (uint32_t)n, 999u);
        uint4* in4=(uint4*)tab; uint4* out4=(uint4*)(tab + (size_t)n*4);   // second half
        float ms = timeit([&]{ k_gather_rec<uint4><<<(n+255)/256,256>>>(in4, idx, out4, n); });
        printf("record gather 16B random: %.3f ms  %.1f Grec/s  alg %.1f GB/s (36 B/rec)\n", ms, n/(ms*1e6), n*36.0/(ms*1e6));
        k_fill_idx<<<(n+255)/256,256>>>(idx, n, (uint32_t)(n/2), 999u); R32* in8=(R32*)tab; R32* out8=(R32*)(tab + (size_t)n*4);
        ms = timeit([&]{ k_gather_rec<R32><<<(n/2+255)/256,256>>>(in8, idx, out8, n/2); });
        printf("record gather 32B random (n/2): %.3f ms  %.1f Grec/s  alg %.1f GB/s (68 B/rec)\n", ms, n/2/(ms*1e6), (n/2)*68.0/(ms*1e6));
        // local-window: sources random within windows of 1M records (16 MB): L2-resident reads
        k_fill_idx<<<(n+255)/256,256>>>(idx, n, 1u<<20, 4242u);
        ms = timeit([&]{ k_gather_rec<uint4><<<(n+255)/256,256>>>(in4, idx, out4, n); });
        printf("record gather 16B from 16MB window: %.3f ms  %.1f Grec/s\n", ms, n/(ms*1e6));
    }
    return 0;
}
