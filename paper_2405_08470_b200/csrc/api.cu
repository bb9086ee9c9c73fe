// C-ABI of libmttkrp_b200 (include/mttkrp.h): argument checks, the layout state machine
// (Alg. 5) and the host-buffer convenience entry point.
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <new>
#include <utility>
#include <vector>
#include "common.cuh"

namespace mk {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}


static mttkrp_status_t check_shape(int nmodes, const int64_t* dims, int64_t nnz) {
    if (!dims) { set_error("dims is NULL"); return MTTKRP_EINVAL; }
    if (nmodes < 2 || nmodes > kMaxModes) { set_error("nmodes %d outside [2,%d]", nmodes, kMaxModes); return MTTKRP_EUNSUPPORTED; }
    for (int m = 0; m < nmodes; ++m) {
        if (dims[m] <= 0) { set_error("dims[%d] = %lld must be positive", m, (long long)dims[m]); return MTTKRP_EINVAL; }
        if (dims[m] >= (1LL << 28)) { set_error("dims[%d] >= 2^28 unsupported", m); return MTTKRP_EUNSUPPORTED; }
    }
    if (nnz < 0) { set_error("nnz < 0"); return MTTKRP_EINVAL; }
    if (nnz >= 0x7fffffffLL) { set_error("nnz >= 2^31 unsupported"); return MTTKRP_EUNSUPPORTED; }
    return MTTKRP_OK;
}

static bool valid_rank(int R) { return R == 8 || R == 16 || R == 32 || R == 64; }
static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int ceil_log2(int64_t x) {
    int b = 0;
    while (((int64_t)1 << b) < x) ++b;
    return b;
}

// Layout state machine (Alg. 5's swap).  d == cur: nothing.  d == cur+1:
// the stored walk (the paper's only case).  Any other d: the stored gather maps of the layouts in
// between are composed into ONE direct map cur -> d (4-byte gathers), cached for the next identical jump, and the
// records move once.  Layouts are absolute orders (remap ids are positions), so the result does
// not depend on the path.
static mttkrp_status_t ensure_layout(mttkrp_handle_s* h, int d, cudaStream_t st) {
    if (h->cur == d) return MTTKRP_OK;
    if (h->alt_layout == d) {                             // the fused kernel of the previous mode already wrote layout d
        uint32_t* t = h->rec_cur;                         // swap(T_in, T_out), Alg. 5 line 12
        h->rec_cur = h->rec_alt;
        h->rec_alt = t;
        h->cur = d;
        h->alt_layout = -1;
        h->remaps_done++;
        return MTTKRP_OK;
    }
    h->alt_layout = -1;                                   // any other pass overwrites the other copy
    const int N = h->N, from = h->cur;
    const int steps = ((d - from) % N + N) % N;
    if (steps == 1 || h->nnz == 0) return launch_remap(h, from, d, nullptr, st);
    if (!(h->jump_map && h->jump_from == from && h->jump_to == d)) {
        // acc_s[j] = position in layout `from` of the element at position j of layout from+s
        const uint32_t* acc = h->mode[from].next;
        for (int s = 1; s < steps; ++s) {
            uint32_t* outb = h->jump[(s - 1) & 1];
            TimedLaunch tl(h->timing, kClsRemap, st);
            MK_TRY(launch_perm_step(h->mode[(from + s) % N].next, acc, outb, h->nnz, st));
            acc = outb;
        }
        h->jump_map = acc;
        h->jump_from = from;
        h->jump_to = d;
    }
    return launch_remap(h, from, d, h->jump_map, st);
}

// Calls on one handle share the two tensor copies and the carry buffer, so they must execute in call order.
// The handle remembers the stream of its last call and an event recorded after it; a call that arrives on a
// different stream first makes that stream wait on the event.
static mttkrp_status_t order_begin(mttkrp_handle_s* h, cudaStream_t st) {
    if (h->launched && st != h->last_stream) MK_CUDA(cudaStreamWaitEvent(st, h->ev_order, 0));
    return MTTKRP_OK;
}
static mttkrp_status_t order_end(mttkrp_handle_s* h, cudaStream_t st) {
    MK_CUDA(cudaEventRecord(h->ev_order, st));
    h->last_stream = st;
    h->launched = 1;
    return MTTKRP_OK;
}

// Mode d on whatever layout is resident: remap passes until the copy is in layout d (the cyclic
// order of Alg. 5 costs one), then the MTTKRP kernels.
static mttkrp_status_t run_mode(mttkrp_handle_s* h, int d, const float* const* factors, int R, float* out, cudaStream_t st) {
    MK_TRY(ensure_layout(h, d, st));
    MK_TRY(launch_mttkrp(h, d, factors, R, out, st));
    if (h->fuse && h->nnz > 0) {                          // the kernel also scattered the records into layout d+1
        const int to = (d + 1) % h->N;
        TimedLaunch tl(h->timing, kClsRemap, st);
        MK_TRY(launch_remap_padding(h, d, to, st));
        h->alt_layout = to;
    }
    return MTTKRP_OK;
}

}  // namespace mk

using namespace mk;

extern "C" {

const char* mttkrp_last_error(void) { return g_err; }
const char* mttkrp_version(void) { return "mttkrp_b200 0.1 sm_100a"; }

mttkrp_status_t mttkrp_workspace_bytes(int nmodes, const int64_t* dims, int64_t nnz, int max_rank, size_t* bytes) {
    if (!bytes) { set_error("bytes is NULL"); return MTTKRP_EINVAL; }
    MK_TRY(check_shape(nmodes, dims, nnz));
    if (max_rank != 0 && !valid_rank(max_rank)) { set_error("max_rank %d not in {0,8,16,32,64}", max_rank); return MTTKRP_EUNSUPPORTED; }
    LayoutPlan lp;
    MK_TRY(plan_layouts(nmodes, dims, nnz, &lp));
    WorkspacePlan p;
    const int sms = device_sm_count();
    MK_TRY(plan_workspace(nmodes, dims, nnz, max_rank, lp.rec_words, sms, lp.policy ? (lp.kappa ? lp.kappa : sms) : 0, lp.fuse, &p));
    *bytes = p.total;
    return MTTKRP_OK;
}

mttkrp_status_t mttkrp_create(mttkrp_handle_t* out, int nmodes, const int64_t* dims, int64_t nnz, const int32_t* idx,
                              const float* vals, int max_rank, void* workspace, size_t workspace_bytes,
                              void* cuda_stream) {
    if (!out) { set_error("out is NULL"); return MTTKRP_EINVAL; }
    *out = nullptr;
    MK_TRY(check_shape(nmodes, dims, nnz));
    if (max_rank != 0 && !valid_rank(max_rank)) { set_error("max_rank %d not in {0,8,16,32,64}", max_rank); return MTTKRP_EUNSUPPORTED; }
    if (nnz > 0 && (!idx || !vals)) { set_error("idx/vals is NULL"); return MTTKRP_EINVAL; }
    if (!workspace) { set_error("workspace is NULL"); return MTTKRP_EWORKSPACE; }
    if (reinterpret_cast<uintptr_t>(workspace) & 255u) { set_error("workspace must be 256-byte aligned"); return MTTKRP_EWORKSPACE; }
    if (nnz > 0 && (!aligned16(idx) || !aligned16(vals))) { set_error("idx/vals must be 16-byte aligned"); return MTTKRP_EINVAL; }
    LayoutPlan lp;
    MK_TRY(plan_layouts(nmodes, dims, nnz, &lp));
    WorkspacePlan p;
    const int num_sms = device_sm_count();
    const int kappa = lp.policy ? (lp.kappa ? lp.kappa : num_sms) : 0;
    MK_TRY(plan_workspace(nmodes, dims, nnz, max_rank, lp.rec_words, num_sms, kappa, lp.fuse, &p));
    if (workspace_bytes < p.total) {
        set_error("workspace %zu bytes < required %zu", workspace_bytes, p.total);
        return MTTKRP_EWORKSPACE;
    }
    int dev = 0;
    MK_CUDA(cudaGetDevice(&dev));

    mttkrp_handle_s* h = new (std::nothrow) mttkrp_handle_s();
    if (!h) { set_error("out of host memory"); return MTTKRP_EINVAL; }
    memset(h, 0, sizeof(*h));
    char* ws = static_cast<char*>(workspace);
    h->N = nmodes;
    h->nnz = nnz;
    for (int m = 0; m < nmodes; ++m) h->dims[m] = dims[m];
    h->rec_words = lp.rec_words;
    h->packed = lp.packed;
    h->shard_nnz = p.shard_nnz;
    h->num_shards = p.num_shards;
    h->policy = lp.policy;
    h->kappa = kappa;
    h->fuse = lp.fuse;
    h->alt_layout = -1;
    h->rec_cur = reinterpret_cast<uint32_t*>(ws + p.rec_a);
    h->rec_alt = reinterpret_cast<uint32_t*>(ws + p.rec_b);
    h->perm0 = reinterpret_cast<uint32_t*>(ws + p.perm0);
    h->carry = reinterpret_cast<float*>(ws + p.carry);
    h->cur = 0;
    h->max_rank = max_rank;
    h->device = dev;
    h->num_sms = num_sms;
    h->knobs = lp.knobs;
    h->force_deep = lp.knobs.force_deep;                          // tests: 0 / 1 pins the kernel variant
    h->jump[0] = reinterpret_cast<uint32_t*>(ws + p.jump[0]);
    h->jump[1] = reinterpret_cast<uint32_t*>(ws + p.jump[1]);
    h->jump_map = nullptr;
    h->jump_from = h->jump_to = -1;
    if (cudaEventCreateWithFlags(&h->ev_order, cudaEventDisableTiming) != cudaSuccess) {
        set_error("cudaEventCreate failed");
        delete h;
        return MTTKRP_ECUDA;
    }
    h->timing = new (std::nothrow) Timing();
    for (int d = 0; d < nmodes; ++d) {
        ModeMeta& mm = h->mode[d];
        for (int l = 0; l < nmodes; ++l) mm.order[l] = lp.order[d][l];
        mm.pk = lp.pk[d];
        for (int l = 0; l < nmodes; ++l) mm.pos[mm.order[l]] = l;
        mm.next = reinterpret_cast<uint32_t*>(ws + p.next[d]);
        mm.ord = reinterpret_cast<uint32_t*>(ws + p.ord[d]);
        mm.osrc = reinterpret_cast<uint32_t*>(ws + p.osrc[d]);
        mm.lflags = reinterpret_cast<uint8_t*>(ws + p.lflags[d]);
        mm.empty_rows = reinterpret_cast<uint32_t*>(ws + p.empty[d]);
        mm.chains = reinterpret_cast<uint32_t*>(ws + p.chains[d]);
        mm.bins = reinterpret_cast<uint32_t*>(ws + p.bins[d]);
        mm.scat = reinterpret_cast<uint32_t*>(ws + p.scat[d]);
        mm.sflags = reinterpret_cast<uint8_t*>(ws + p.sflags[d]);
        if (max_rank > 0) {
            h->stage_fac[d] = reinterpret_cast<float*>(ws + p.stage_fac[d]);
            h->stage_out[d] = reinterpret_cast<float*>(ws + p.stage_out[d]);
        }
    }
    h->bytes_held = (int64_t)p.total;                             // until build_format has chosen the walks
    mttkrp_status_t s = build_format(h, p, ws, idx, vals, static_cast<cudaStream_t>(cuda_stream));
    if (s != MTTKRP_OK) { cudaEventDestroy(h->ev_order); delete h->timing; delete h; return s; }
    order_end(h, static_cast<cudaStream_t>(cuda_stream));
    *out = h;
    return MTTKRP_OK;
}

static mttkrp_status_t check_mode_args(mttkrp_handle_t h, int d, const float* const* factors, int R, const float* out) {
    if (!h) { set_error("handle is NULL"); return MTTKRP_EINVAL; }
    if (d < 0 || d >= h->N) { set_error("mode %d outside [0,%d)", d, h->N); return MTTKRP_EINVAL; }
    if (!valid_rank(R)) { set_error("unsupported rank %d (8, 16, 32, 64)", R); return MTTKRP_EUNSUPPORTED; }
    if (!factors || !out) { set_error("factors/out is NULL"); return MTTKRP_EINVAL; }
    if (!aligned16(out)) { set_error("out must be 16-byte aligned"); return MTTKRP_EINVAL; }
    for (int m = 0; m < h->N; ++m) {
        if (m == d) continue;
        if (!factors[m]) { set_error("factors[%d] is NULL", m); return MTTKRP_EINVAL; }
        if (!aligned16(factors[m])) { set_error("factors[%d] must be 16-byte aligned", m); return MTTKRP_EINVAL; }
        if (factors[m] == out) { set_error("out aliases factors[%d]", m); return MTTKRP_EINVAL; }
    }
    return MTTKRP_OK;
}

mttkrp_status_t mttkrp_mode(mttkrp_handle_t h, int d, const float* const* factors, int R, float* out, void* cuda_stream) {
    MK_TRY(check_mode_args(h, d, factors, R, out));
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    MK_TRY(order_begin(h, st));
    const mttkrp_status_t s = run_mode(h, d, factors, R, out, st);
    MK_TRY(order_end(h, st));
    return s;
}

mttkrp_status_t mttkrp_sweep(mttkrp_handle_t h, const float* const* factors, int R, float* const* outs, void* cuda_stream) {
    if (!h) { set_error("handle is NULL"); return MTTKRP_EINVAL; }
    if (!outs) { set_error("outs is NULL"); return MTTKRP_EINVAL; }
    for (int d = 0; d < h->N; ++d) MK_TRY(check_mode_args(h, d, factors, R, outs[d]));
    for (int d = 0; d < h->N; ++d) MK_TRY(mttkrp_mode(h, d, factors, R, outs[d], cuda_stream));
    return MTTKRP_OK;
}

mttkrp_status_t mttkrp_remap_to(mttkrp_handle_t h, int d, void* cuda_stream) {
    if (!h) { set_error("handle is NULL"); return MTTKRP_EINVAL; }
    if (d < 0 || d >= h->N) { set_error("mode %d outside [0,%d)", d, h->N); return MTTKRP_EINVAL; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    MK_TRY(order_begin(h, st));
    const mttkrp_status_t s = ensure_layout(h, d, st);
    MK_TRY(order_end(h, st));
    return s;
}

mttkrp_status_t mttkrp_sweep_host(mttkrp_handle_t h, const float* const* factors, int R, float* const* outs,
                                  void* cuda_stream) {
    if (!h) { set_error("handle is NULL"); return MTTKRP_EINVAL; }
    if (!valid_rank(R)) { set_error("unsupported rank %d (8, 16, 32, 64)", R); return MTTKRP_EUNSUPPORTED; }
    if (R > h->max_rank) { set_error("R %d > max_rank %d given at create", R, h->max_rank); return MTTKRP_EINVAL; }
    if (!factors || !outs) { set_error("factors/outs is NULL"); return MTTKRP_EINVAL; }
    for (int m = 0; m < h->N; ++m)
        if (!factors[m] || !outs[m]) { set_error("factors[%d]/outs[%d] is NULL", m, m); return MTTKRP_EINVAL; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (!h->host_path_ready) {
        MK_CUDA(cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking));
        MK_CUDA(cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking));
        for (int m = 0; m < h->N; ++m) {
            MK_CUDA(cudaEventCreateWithFlags(&h->ev_in[m], cudaEventDisableTiming));
            MK_CUDA(cudaEventCreateWithFlags(&h->ev_done[m], cudaEventDisableTiming));
        }
        MK_CUDA(cudaEventCreateWithFlags(&h->ev_sync, cudaEventDisableTiming));
        h->host_path_ready = 1;
    }
    // Copies overlap the kernels: factors go in on one stream (A_0, which mode 0 does not read, last), every
    // Y_d goes out on another while the next mode runs; the caller's stream carries the kernels.
    const float* dfac[kMaxModes];
    MK_TRY(order_begin(h, st));
    MK_CUDA(cudaEventRecord(h->ev_sync, st));
    MK_CUDA(cudaStreamWaitEvent(h->s_in, h->ev_sync, 0));
    for (int i = 0; i < h->N; ++i) {
        const int m = (i + 1) % h->N;
        MK_CUDA(cudaMemcpyAsync(h->stage_fac[m], factors[m], (size_t)h->dims[m] * R * 4, cudaMemcpyHostToDevice, h->s_in));
        MK_CUDA(cudaEventRecord(h->ev_in[m], h->s_in));
        dfac[m] = h->stage_fac[m];
    }
    for (int d = 0; d < h->N; ++d) {
        if (d == 0) {
            for (int m = 1; m < h->N; ++m) MK_CUDA(cudaStreamWaitEvent(st, h->ev_in[m], 0));
        } else if (d == 1) {
            MK_CUDA(cudaStreamWaitEvent(st, h->ev_in[0], 0));
        }
        MK_TRY(run_mode(h, d, dfac, R, h->stage_out[d], st));
        MK_CUDA(cudaEventRecord(h->ev_done[d], st));
        MK_CUDA(cudaStreamWaitEvent(h->s_out, h->ev_done[d], 0));
        MK_CUDA(cudaMemcpyAsync(outs[d], h->stage_out[d], (size_t)h->dims[d] * R * 4, cudaMemcpyDeviceToHost, h->s_out));
    }
    MK_TRY(order_end(h, st));
    MK_CUDA(cudaStreamSynchronize(st));
    MK_CUDA(cudaStreamSynchronize(h->s_out));
    return MTTKRP_OK;
}

mttkrp_status_t mttkrp_destroy(mttkrp_handle_t h) {
    if (!h) { set_error("handle is NULL"); return MTTKRP_EINVAL; }
    // The workspace goes back to the caller: wait until the handle's last launched work has finished with it.
    if (h->launched) cudaEventSynchronize(h->ev_order);
    cudaEventDestroy(h->ev_order);
    if (h->timing) {
        for (auto& e : h->timing->ev) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
        delete h->timing;
    }
    if (h->host_path_ready) {
        for (int m = 0; m < h->N; ++m) { cudaEventDestroy(h->ev_in[m]); cudaEventDestroy(h->ev_done[m]); }
        cudaEventDestroy(h->ev_sync);
        cudaStreamDestroy(h->s_in);
        cudaStreamDestroy(h->s_out);
    }
    delete h;
    return MTTKRP_OK;
}

mttkrp_status_t mttkrp_timing_begin(mttkrp_handle_t h) {
    if (!h || !h->timing) { set_error("handle is NULL"); return MTTKRP_EINVAL; }
    for (auto& e : h->timing->ev) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    h->timing->ev.clear();
    h->timing->on = true;
    return MTTKRP_OK;
}

mttkrp_status_t mttkrp_timing_end(mttkrp_handle_t h, mttkrp_timing_t* out, void* cuda_stream) {
    if (!h || !h->timing || !out) { set_error("handle/out is NULL"); return MTTKRP_EINVAL; }
    h->timing->on = false;
    memset(out, 0, sizeof(*out));
    MK_CUDA(cudaStreamSynchronize(static_cast<cudaStream_t>(cuda_stream)));
    double ms[4] = {0, 0, 0, 0};
    int64_t cnt[4] = {0, 0, 0, 0};
    for (auto& e : h->timing->ev) {
        float t = 0.f;
        MK_CUDA(cudaEventSynchronize(e.b));
        MK_CUDA(cudaEventElapsedTime(&t, e.a, e.b));
        ms[e.cls] += t;
        cnt[e.cls]++;
        cudaEventDestroy(e.a);
        cudaEventDestroy(e.b);
    }
    h->timing->ev.clear();
    out->remap_ms = ms[0]; out->zero_ms = ms[1]; out->mttkrp_ms = ms[2]; out->fixup_ms = ms[3];
    out->remap_launches = cnt[0]; out->zero_launches = cnt[1]; out->mttkrp_launches = cnt[2]; out->fixup_launches = cnt[3];
    return MTTKRP_OK;
}

mttkrp_status_t mttkrp_get_info(mttkrp_handle_t h, mttkrp_info_t* info) {
    if (!h || !info) { set_error("handle/info is NULL"); return MTTKRP_EINVAL; }
    memset(info, 0, sizeof(*info));
    info->nmodes = h->N;
    info->cur_layout = h->cur;
    info->nnz = h->nnz;
    int64_t bits = 32;
    for (int m = 0; m < h->N; ++m) {
        info->dims[m] = h->dims[m];
        info->num_split_rows[m] = h->mode[m].n_chains;
        info->num_empty_rows[m] = h->mode[m].n_empty;
        for (int l = 0; l < h->N; ++l) info->key_order[m][l] = h->mode[m].order[l];
        info->remap_blocked[m] = h->mode[m].blocked;
        info->remap_avg_run[m] = h->mode[m].avg_run;
        bits += ceil_log2(h->dims[m]);
    }
    bits += (int64_t)h->N * ceil_log2(h->nnz > 1 ? h->nnz : 2);
    info->record_bytes = 4 * h->rec_words;
    info->shard_nnz = h->shard_nnz;
    info->num_shards = h->num_shards;
    info->bytes_held = h->bytes_held;
    info->bytes_paper_format = (h->nnz * bits + 7) / 8;
    info->remaps_done = h->remaps_done;
    for (int m = 0; m < h->N; ++m) { info->remap_plain_ms[m] = h->mode[m].plain_ms; info->remap_twopass_ms[m] = h->mode[m].twopass_ms; }
    info->fused_remap = h->fuse;
    for (int m = 0; m < h->N; ++m) { info->cold_rows[m] = h->cold_rows[m]; info->cold_degree[m] = (int64_t)h->cold_deg[m]; }
    info->shard_policy = h->policy;
    info->kappa = h->kappa;
    for (int m = 0; m < h->N; ++m) { info->max_partition_nnz[m] = h->mode[m].max_bin; info->min_partition_nnz[m] = h->mode[m].min_bin; }
    return MTTKRP_OK;
}

mttkrp_status_t mttkrp_get_perm(mttkrp_handle_t h, int d, uint32_t* perm_dev, uint32_t* scratch_dev, void* cuda_stream) {
    if (!h) { set_error("handle is NULL"); return MTTKRP_EINVAL; }
    if (d < 0 || d >= h->N) { set_error("mode %d outside [0,%d)", d, h->N); return MTTKRP_EINVAL; }
    if (h->nnz == 0) return MTTKRP_OK;
    if (!perm_dev || (d > 0 && !scratch_dev)) { set_error("perm/scratch is NULL"); return MTTKRP_EINVAL; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    MK_TRY(order_begin(h, st));
    // perm_{j+1}[k] = perm_j[next_j[k]]; choose the start buffer so that step d lands in perm_dev.
    uint32_t* a = (d % 2 == 0) ? perm_dev : scratch_dev;
    uint32_t* b = (d % 2 == 0) ? scratch_dev : perm_dev;
    MK_CUDA(cudaMemcpyAsync(a, h->perm0, (size_t)h->nnz * 4, cudaMemcpyDeviceToDevice, st));
    for (int j = 0; j < d; ++j) {
        MK_TRY(launch_perm_step(h->mode[j].next, a, b, h->nnz, st));
        uint32_t* t = a; a = b; b = t;
    }
    return order_end(h, st);
}

mttkrp_status_t mttkrp_export_coo(mttkrp_handle_t h, int32_t* idx_dev, float* vals_dev, void* cuda_stream) {
    if (!h) { set_error("handle is NULL"); return MTTKRP_EINVAL; }
    if (h->nnz == 0) return MTTKRP_OK;
    if (!idx_dev || !vals_dev) { set_error("idx/vals is NULL"); return MTTKRP_EINVAL; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    MK_TRY(order_begin(h, st));
    MK_TRY(launch_export(h, idx_dev, vals_dev, st));
    return order_end(h, st);
}

mttkrp_status_t mttkrp_partition_rows(mttkrp_handle_t h, int d, int kappa, int32_t* deg_dev, int32_t* part_of_row,
                                      int64_t* loads, void* cuda_stream) {
    if (!h) { set_error("handle is NULL"); return MTTKRP_EINVAL; }
    if (d < 0 || d >= h->N) { set_error("mode %d outside [0,%d)", d, h->N); return MTTKRP_EINVAL; }
    if (kappa < 1) { set_error("kappa %d < 1", kappa); return MTTKRP_EINVAL; }
    if (!deg_dev || !loads) { set_error("deg_dev/loads is NULL"); return MTTKRP_EINVAL; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    MK_TRY(order_begin(h, st));
    MK_TRY(launch_row_degrees(h, d, deg_dev, st));
    MK_TRY(order_end(h, st));
    const int64_t rows = h->dims[d];
    std::vector<int32_t> deg;
    try { deg.resize((size_t)rows); } catch (...) { set_error("mttkrp_partition_rows: out of host memory"); return MTTKRP_EINVAL; }
    MK_CUDA(cudaMemcpyAsync(deg.data(), deg_dev, sizeof(int32_t) * (size_t)rows, cudaMemcpyDeviceToHost, st));
    MK_CUDA(cudaStreamSynchronize(st));
    if (!lpt_partition(deg.data(), rows, kappa, part_of_row, loads)) {
        set_error("mttkrp_partition_rows: out of host memory");
        return MTTKRP_EINVAL;
    }
    return MTTKRP_OK;
}

}  // extern "C"
