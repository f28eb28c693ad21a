// =====================================================================================
// ng.cu — host side of libng.so: the C-ABI declared in include/ng.h.
//
// Holds the population table and the list of connect calls, runs the on-device connection builder
// (ng_prepare) and enqueues the per-step kernels of ng_device.cuh (ng_simulate), either as a replayed CUDA
// graph of `steps_per_graph` steps, as plain launches, or as one persistent cooperative kernel.
//
// Update/deliver handshake without host round trips: update(n) reads ctl.step_u and writes ctl.step_d;
// deliver(n) reads ctl.step_d and ctl.spike_cnt[n&1], and one of its threads writes ctl.step_u = n+1 and
// clears ctl.spike_cnt[(n+1)&1].  Each kernel only reads words the other kind of kernel writes, so a captured
// graph replays unchanged for any step index.
//
// No CPU fallback exists: every entry point that computes needs a CUDA device and fails with NG_ERR_CUDA otherwise.
// =====================================================================================
#include "../../include/ng.h"
#include "ng_device.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

using namespace ng;

struct HostPop { int32_t first, n; ng_lif_params p; PopDev dev; };     // dev.model tells LIF from AdEx

struct ng_sim {
    ng_config cfg{};
    ng_allocator alloc{};
    bool has_alloc = false;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    std::string err;
    std::vector<HostPop> pops;
    std::vector<CallDev> calls;
    int32_t N = 0;
    int64_t S = 0;
    bool prepared = false;
    int32_t bypass = 0; uint32_t inject_thr = 0;
    // options
    int list_bufs = 2;
    int step_kernel = 0;
    int step_mode_opt = 3; int step_mode = 0; int steps_per_graph = 100; int delivery_kernel_opt = 0; int deliver_blocks_opt = 0;
    bool trace_on = false; unsigned long long* trace_saved = nullptr; int last_persistent_blocks = 0;
    int profile = 0; int async = 0; int sort_segments = 1; int prefetch_opt = 1;
    // device
    std::vector<void*> allocs;
    StepArgs a{};
    uint32_t* d_cnt = nullptr; long long* d_row_len = nullptr; long long* d_row_off = nullptr;
    uint32_t* d_grp_rel = nullptr; int32_t* d_tgt = nullptr; float* d_w = nullptr; uint8_t* d_dly = nullptr;
    RowInfo* d_row_info = nullptr;
    CallDev* d_calls = nullptr; PopDev* d_pops = nullptr; uint8_t* d_pop_of = nullptr; Ctl* d_ctl = nullptr;
    int64_t n_padded = 0; int64_t max_row_records = 0;
    int sm_count = 148; size_t l2_bytes = 0; bool coop_ok = false;
    int delivery_kernel = 1; int deliver_blocks = 0; int update_blocks = 0; int persistent_blocks = 0;
    int pipe_blocks = 0; int persistent_pipe_blocks = 0;
    int persistent_threads = kPersistentThreads;
    // statistics (ng_enable_statistics)
    int32_t* d_st_sample = nullptr; int st_sample_per_pop = 0; int st_slots = 0;
    bool one_round_step = false, one_round_persistent = false;   // the network is covered in one round of updater threads
    size_t resm_bytes = 0;                 // > 0: multi-round LIF network with its state resident in dynamic shared memory (kResM)
    bool has_adex = false;                 // any AdEx population: two receptor ports, AdEx state arrays, <true> kernels
    int64_t NR = 0;                        // ring row length = N * ports
    bool window_backend = false;           // delivery kernel 4 or 6 chosen before ng_prepare: spike window instead of a D-plane ring
    bool pipewin = false;                  //   6: the window walked by the rest warps of the pipelined persistent kernel
    // target-sharded multi-GPU (ng_set_shard): this handle owns the neurons [id_first, id_first + NL)
    int shard_rank = 0, shard_world = 1; int32_t id_first = 0; int32_t NL = 0;
    unsigned char* xchg_own = nullptr; size_t xchg_bytes = 0; bool xchg_ipc_open[16] = {};
    bool queue_backend = false;            // delivery kernel 5 chosen before / by ng_prepare: per-delay event queues, two planes
    int64_t queue_cap_opt = 0;             // NG_OPT_QUEUE_CAPACITY: events per queue (0 = auto)
    int queue_blocks = 0;
    cudaGraphExec_t graph_exec = nullptr; int graph_steps = 0;
    // stats
    double build_ms = 0, ms_update = 0, ms_deliver = 0;
    uint64_t launches_update = 0, launches_deliver = 0, launches_other = 0;
    uint64_t rec_dropped = 0;
    uint64_t steps_done = 0;
};

namespace {

int32_t fail(ng_sim* s, int32_t code, const std::string& msg) {
    if (s) s->err = msg;
    return code;
}
#define NG_CUDA(s, expr)                                                                              \
    do {                                                                                              \
        cudaError_t e_ = (expr);                                                                      \
        if (e_ != cudaSuccess)                                                                        \
            return fail((s), e_ == cudaErrorMemoryAllocation ? NG_ERR_OOM : NG_ERR_CUDA,              \
                        std::string(#expr) + ": " + cudaGetErrorString(e_));                          \
    } while (0)

void* dev_alloc(ng_sim* s, size_t bytes) {
    if (bytes == 0) bytes = 256;
    void* p = nullptr;
    if (s->has_alloc) p = s->alloc.alloc(bytes, s->alloc.user);
    else if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); p = nullptr; }
    if (p) s->allocs.push_back(p);
    return p;
}
void dev_free(ng_sim* s, void* p) {
    if (!p) return;
    auto it = std::find(s->allocs.begin(), s->allocs.end(), p);
    if (it != s->allocs.end()) s->allocs.erase(it);
    if (s->has_alloc) s->alloc.free(p, s->alloc.user);
    else cudaFree(p);
}
template <typename T>
bool dev_alloc_t(ng_sim* s, T** out, size_t count) {
    *out = (T*)dev_alloc(s, count * sizeof(T));
    return *out != nullptr;
}

// Exact-integration propagators of PAPER.md Eqs. (1)-(2) over one step h (ref. 20), fp64:
// x = (I, V - E_L), dx/dt = A x, A = [[-1/tau_syn, 0], [1/C_m, -1/tau_m]]; exp(A h) = [[P11, 0], [P21, P22]].
void make_pop_dev(const ng_lif_params& p, double h, PopDev& d) {
    const double P11 = std::exp(-h / p.tau_syn);
    const double P22 = std::exp(-h / p.tau_m);
    const double P21 = p.tau_m * p.tau_syn / (p.C_m * (p.tau_m - p.tau_syn)) * (P22 - P11);
    const double P20 = p.tau_m / p.C_m * (1.0 - P22);
    d.P11 = (float)P11; d.P22 = (float)P22; d.P21 = (float)P21; d.P20Ie = (float)(P20 * p.I_e);
    d.E_L = (float)p.E_L; d.V_th = (float)p.V_th; d.V_reset = (float)p.V_reset; d.w_ext = (float)p.poisson_weight;
    d.refr_steps = (int32_t)std::floor(p.t_ref_ms / h + 0.5);
}

// DESIGN.md C7: T[m] = floor(CDF_Poisson(lambda)(m) * 2^32), saturating at 2^32-1, with the pmf recurrence
// p_0 = exp(-lambda), p_{m+1} = (p_m * lambda) / (m+1), CDF accumulated in that order in fp64.
bool make_poisson_table(double lam, PopDev& d) {
    d.n_T = 0;
    if (!(lam > 0.0)) return true;
    double p = std::exp(-lam), c = p;
    for (int m = 0; m < kMaxPoissonTable; ++m) {
        const double s = std::floor(c * 4294967296.0);
        const uint32_t t = s >= 4294967295.0 ? 4294967295u : (uint32_t)s;
        d.T[d.n_T++] = t;
        if (t == 4294967295u) return true;
        const double pl = p * lam;
        p = pl / (double)(m + 1);
        c = c + p;
    }
    return false;
}

bool valid_dist(const ng_dist* d) {
    return d && d->kind >= NG_DIST_CONST && d->kind <= NG_DIST_UNIFORM_INT;
}

int32_t add_call(ng_sim* s, int32_t rule, int32_t src_first, int32_t src_n, int32_t tgt_first, int32_t tgt_n, int32_t K,
                 const ng_dist* w, const ng_dist* d, int32_t port = 0) {
    if (!s) return NG_ERR_INVALID_ARG;
    if (s->prepared) return fail(s, NG_ERR_STATE, "connect after ng_prepare");
    if (!valid_dist(w) || !valid_dist(d)) return fail(s, NG_ERR_INVALID_ARG, "bad distribution");
    if (src_n <= 0 || tgt_n <= 0 || K < 0 || src_first < 0 || tgt_first < 0 ||
        (int64_t)src_first + src_n > s->N || (int64_t)tgt_first + tgt_n > s->N)
        return fail(s, NG_ERR_INVALID_ARG, "population range outside the created neurons, or K < 0");
    CallDev c{};
    c.rule = rule; c.src_first = src_first; c.src_n = src_n; c.tgt_first = tgt_first; c.tgt_n = tgt_n; c.K = K;
    if (port < 0 || port > 1) return fail(s, NG_ERR_INVALID_ARG, "receptor port is 0 or 1");
    c.call_index = (int32_t)s->calls.size(); c.port = port;
    c.w = DistDev{w->kind, 0, w->a, w->b, w->lo, w->hi};
    c.d = DistDev{d->kind, 0, d->a, d->b, d->lo, d->hi};
    s->calls.push_back(c);
    return NG_OK;
}

int grid_for(long long work, int threads, int cap) {
    long long b = (work + threads - 1) / threads;
    if (b < 1) b = 1;
    if (b > cap) b = cap;
    return (int)b;
}

void destroy_graph(ng_sim* s) {
    if (s->graph_exec) { cudaGraphExecDestroy(s->graph_exec); s->graph_exec = nullptr; s->graph_steps = 0; }
}

void launch_update(ng_sim* s) {
    if (s->has_adex) update_kernel<true><<<s->update_blocks, kUpdateThreads, 0, s->stream>>>(s->a);
    else update_kernel<false><<<s->update_blocks, kUpdateThreads, 0, s->stream>>>(s->a);
}
void launch_deliver(ng_sim* s) {
    if (s->delivery_kernel == 5) queue_deliver_kernel<<<s->queue_blocks, kQThreads, 0, s->stream>>>(s->a);
    else if (s->delivery_kernel == 4) deliver_kernel<4><<<s->deliver_blocks, kDeliverThreads, 0, s->stream>>>(s->a);
    else if (s->delivery_kernel == 2) deliver_kernel<2><<<s->deliver_blocks, kDeliverThreads, 0, s->stream>>>(s->a);
    else deliver_kernel<1><<<s->deliver_blocks, kDeliverThreads, 0, s->stream>>>(s->a);
}

// one time step: two kernels (update, deliver) or the pipelined step kernel
void launch_pipe(ng_sim* s) {
    if (s->has_adex && s->one_round_step) pipe_step_kernel<true, true, true><<<s->pipe_blocks, kPipeThreads, 0, s->stream>>>(s->a);
    else if (s->has_adex) pipe_step_kernel<true, true, false><<<s->pipe_blocks, kPipeThreads, 0, s->stream>>>(s->a);
    else if (s->one_round_step) pipe_step_kernel<true, false, true><<<s->pipe_blocks, kPipeThreads, 0, s->stream>>>(s->a);
    else pipe_step_kernel<true, false, false><<<s->pipe_blocks, kPipeThreads, 0, s->stream>>>(s->a);
}
// rest pass of the last step of an ng_simulate call (pipelined delivery kernel 3): leaves nothing pending between API calls
void launch_pipe_flush(ng_sim* s) {
    if (s->has_adex) pipe_step_kernel<false, true><<<s->pipe_blocks, kPipeThreads, 0, s->stream>>>(s->a);
    else pipe_step_kernel<false, false><<<s->pipe_blocks, kPipeThreads, 0, s->stream>>>(s->a);
}
void launch_exchange_publish(ng_sim* s) { xchg_publish_kernel<<<s->shard_world, 256, 0, s->stream>>>(s->a); }
void launch_exchange_gather(ng_sim* s) { xchg_gather_kernel<<<s->shard_world, 256, 0, s->stream>>>(s->a); }
void launch_step(ng_sim* s) {
    if (s->delivery_kernel == 3) launch_pipe(s);
    else if (s->shard_world > 1) { launch_update(s); launch_exchange_publish(s); launch_exchange_gather(s); launch_deliver(s); }
    else { launch_update(s); launch_deliver(s); }
}
// choose launch shapes from the built network (static per simulation; no per-step host decisions)
void configure_launch(ng_sim* s) {
    const int sm = s->sm_count;
    s->update_blocks = grid_for(s->NL, kUpdateThreads, sm * 32);
    // delivery kernel: delay-major segment walk pays off when the ring is too big to stay in L2 next to the
    // streamed records and groups are long enough to fill a warp's 128-bit loads; otherwise walk whole rows.
    const double ring_bytes = (double)s->N * s->cfg.ring_slots * 4.0;
    const double mean_group = s->N > 0 ? (double)s->S / ((double)s->N * s->cfg.ring_slots) : 0.0;
    int k = s->delivery_kernel_opt;
    // otherwise the step is latency-bound: rows are walked whole (kernel 1) or by the pipelined step kernel (3).
    if (k == 0) k = s->shard_world > 1 ? 1 : 3;                     // a ring beyond L2 was given a two-plane backend in ng_prepare
    if (k == 3 && s->shard_world > 1) k = 1;                        // the pipelined kernel delivers a CTA's own spikes: one GPU only
    (void)mean_group; (void)ring_bytes;
    if (s->window_backend) k = s->pipewin ? 6 : 4;                  // fixed at ng_prepare: there is no D-plane ring
    if (s->queue_backend) k = 5;
    s->delivery_kernel = k;
    // step mode: the latency-bound kernels run as one persistent cooperative kernel per ng_simulate call; the
    // bandwidth-bound delay-major kernel keeps its 8 CTAs per SM and runs from a CUDA graph
    s->step_mode = s->step_mode_opt != 3 ? s->step_mode_opt : (k == 2 || k == 4 || k == 5 || !s->coop_ok) ? 0 : 2;
    if (s->has_adex && s->step_mode == 2 && k != 3 && k != 6) s->step_mode = 0;   // the two-phase persistent kernels are LIF only
    if (k == 6) s->step_mode = 2;                                       // exists as a persistent cooperative kernel only
    if (k == 5 && s->step_mode == 2) s->step_mode = 0;                  // the event-queue backend runs as update + delivery launches
    if (s->shard_world > 1 && s->step_mode == 2) s->step_mode = 0;      // sharded: update, exchange and delivery are separate launches
    s->a.prefetch = (k != 2 && k != 4 && k != 5 && s->prefetch_opt) ? 1 : 0;      // (kernel 6: the delay-1 head only)
    {
        int occq = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occq, queue_deliver_kernel, kQThreads, 0);
        s->queue_blocks = sm * std::max(1, std::min(occq, 1024 / kQThreads));
    }
    s->pipe_blocks = grid_for(s->N, kPipeThreads - (s->has_adex ? kAdexRest : kEntryTile), sm * 4);   // updaters per CTA
    {
        int occp = 0;
        const int pt = s->has_adex ? 512 : s->persistent_threads;      // AdEx kernels are compiled for 512-thread CTAs
        if (s->has_adex) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occp, persistent_pipe_kernel<true, false>, pt, 0);
        else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occp, persistent_pipe_kernel<false, false>, pt, 0);
        if (occp < 1) occp = 1;
        s->persistent_pipe_blocks = sm * std::min(occp, kPersistentThreads / pt);
        // updater threads per CTA of the AdEx kernels: all but four warps (pipe_updater_threads in ng_device.cuh)
        s->one_round_persistent = (long long)s->persistent_pipe_blocks * (pt - (s->has_adex ? kAdexRest : (pt >= 512 ? kEntryTile : 64))) >= s->N;
        // AdEx: the two-pass update (one integration attempt per lane, the unfinished neurons — on the exponential
        // upswing, up to thirty sub-steps — finished by dense warps from a CTA list) pays for any number of rounds:
        // 10^6 neurons 116 -> 105 us per step (profiles/r02_adex1m.md)
        if (s->has_adex) s->one_round_persistent = true;
        s->one_round_step = (long long)s->pipe_blocks * (kPipeThreads - (s->has_adex ? kAdexRest : kEntryTile)) >= s->N;
        // several rounds per step (config 4): keep V, I_syn, refr and the population byte (13 B per neuron) of the CTA's
        // neurons in dynamic shared memory for the whole launch if that fits beside the static 45 KB
        s->resm_bytes = 0;
        if (!s->has_adex && !s->bypass && !s->one_round_persistent && pt - kResMRest >= 256 && s->N > 0) {
            const long long U = pt - kResMRest, per_round = (long long)s->persistent_pipe_blocks * U;
            const long long rounds = (s->N + per_round - 1) / per_round;
            const size_t bytes = ((size_t)(rounds * U) * 13 + 15) & ~(size_t)15;
            int occ2 = 0;
            if (bytes <= 160 * 1024 &&
                cudaFuncSetAttribute(persistent_pipe_kernel<false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) == cudaSuccess &&
                cudaFuncSetAttribute(persistent_pipe_kernel<false, false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) == cudaSuccess &&
                cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, persistent_pipe_kernel<false, false, true>, pt, bytes) == cudaSuccess &&
                (long long)occ2 * s->sm_count >= s->persistent_pipe_blocks)
                s->resm_bytes = bytes;
            cudaGetLastError();
        }
    }
    int blocks = s->deliver_blocks_opt;
    if (blocks <= 0) {
        // enough warps to cover the expected items of a step, between one and eight CTAs per SM
        const double mean_row = s->N > 0 ? (double)s->n_padded / s->N : 0.0;
        const double work_warps = std::max(1.0, mean_row / kChunkRecords) * std::max(1.0, s->N * 0.002);
        long long b = (long long)(work_warps / (kDeliverThreads / 32)) + 1;
        b = ((b + sm - 1) / sm) * sm;
        blocks = (int)std::min<long long>(std::max<long long>(b, sm), (long long)sm * 8);
    }
    s->deliver_blocks = blocks;
    s->a.max_row_chunks = (int32_t)((s->max_row_records + kChunkRecords - 1) / kChunkRecords);
    if (s->a.max_row_chunks < 1) s->a.max_row_chunks = 1;
    s->a.mean_row_records = (int32_t)std::max<int64_t>(1, s->N > 0 ? s->n_padded / s->N : 1);
    // persistent kernel: one CTA of persistent_threads per SM slot; few CTAs keep the grid barrier cheap
    int occ = 0;
    if (s->delivery_kernel == 4) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, persistent_kernel<4>, s->persistent_threads, 0);
    else if (s->delivery_kernel == 2) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, persistent_kernel<2>, s->persistent_threads, 0);
    else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, persistent_kernel<1>, s->persistent_threads, 0);
    if (occ < 1) occ = 1;
    s->persistent_blocks = sm * std::min(occ, kPersistentThreads / s->persistent_threads);
    destroy_graph(s);
}

// Resident one-round LIF networks: the split kernel (persistent_split_kernel: spike decisions a step ahead, list / plane
// barriers, decoupled warp groups) instead of the pipelined kernel with one grid barrier per step?  Yes as soon as every CTA
// holds a neuron (config 0, five neurons per CTA: 2.50 -> 2.38 us per step; the kEarly form of the one-barrier kernel, kept
// behind -DNG_SPLIT_KERNEL=0, only paid from 32 neurons per CTA on: 2.52 -> 2.55-2.68 us at config 0).
#ifndef NG_SPLIT_KERNEL
#define NG_SPLIT_KERNEL 1
#endif
#ifndef NG_EARLY_MIN_PER_CTA
#define NG_EARLY_MIN_PER_CTA (NG_SPLIT_KERNEL ? 1 : 32)
#endif
bool early_decision(const ng_sim* s) {
    return !s->has_adex && s->list_bufs == 4 && (long long)s->N >= (long long)NG_EARLY_MIN_PER_CTA * s->persistent_pipe_blocks;
}

int32_t build_graph(ng_sim* s, int steps) {
    destroy_graph(s);
    cudaGraph_t graph = nullptr;
    NG_CUDA(s, cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal));
    for (int i = 0; i < steps; ++i) launch_step(s);
    NG_CUDA(s, cudaStreamEndCapture(s->stream, &graph));
    cudaError_t e = cudaGraphInstantiate(&s->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) return fail(s, NG_ERR_CUDA, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e));
    s->graph_steps = steps;
    return NG_OK;
}

int32_t read_ctl(ng_sim* s, Ctl* out) {
    NG_CUDA(s, cudaMemcpyAsync(out, s->d_ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s->stream));
    NG_CUDA(s, cudaStreamSynchronize(s->stream));
    return NG_OK;
}

int32_t field_info(ng_sim* s, int32_t field, void** base, size_t* elem, int64_t* len) {
    switch (field) {
        case NG_FIELD_V: *base = s->a.V; *elem = 4; *len = s->NL; return NG_OK;
        case NG_FIELD_I_SYN: *base = s->a.I; *elem = 4; *len = s->NL; return NG_OK;
        case NG_FIELD_REFR: *base = s->a.refr; *elem = 4; *len = s->NL; return NG_OK;
        case NG_FIELD_RING: *base = s->a.ring; *elem = 4; *len = s->NR * s->cfg.ring_slots; return NG_OK;   // see ring_copy
        case NG_FIELD_LAST_INPUT:
            if (!s->a.last_input) return fail(s, NG_ERR_STATE, "NG_FIELD_LAST_INPUT needs NG_DEBUG_INPUT");
            *base = s->a.last_input; *elem = 4; *len = s->NR; return NG_OK;
        case NG_FIELD_ADEX_W: case NG_FIELD_ADEX_G_EX: case NG_FIELD_ADEX_Y_EX: case NG_FIELD_ADEX_G_IN: case NG_FIELD_ADEX_Y_IN:
        case NG_FIELD_ADEX_H: {
            if (!s->has_adex) return fail(s, NG_ERR_STATE, "no AdEx population");
            float* arr[] = {s->a.ax_w, s->a.ax_gx, s->a.ax_yx, s->a.ax_gi, s->a.ax_yi, s->a.ax_h};
            *base = arr[field - NG_FIELD_ADEX_W]; *elem = 4; *len = s->NL; return NG_OK;
        }
        default: return fail(s, NG_ERR_INVALID_ARG, "unknown field");
    }
}

// NG_FIELD_RING as the C-ABI shows it is [D][N], slot s holding the input of the one pending step n' in [n, n+D) with
// n' mod D == s (n = index of the next step).  The device stores Dr = D + 1 planes indexed n' mod Dr (see
// neuron_early in ng_device.cuh); this copies the element range [first, first+count) of the API view plane by plane.
int32_t ring_copy(ng_sim* s, bool to_device, void* user, int64_t count, int64_t first) {
    Ctl h{};
    int32_t rc = read_ctl(s, &h);
    if (rc) return rc;
    const int64_t N = s->NR, D = s->cfg.ring_slots, Dr = s->a.Dr, n = h.step_u;      // N: plane length (all ports)
    if (s->window_backend || s->queue_backend) {
        // no ring exists: the pending inputs live in the spike window / the event queues.  Read-back expands them into a temporary image.
        if (to_device) return fail(s, NG_ERR_STATE, "NG_FIELD_RING cannot be set with the two-plane backends (delivery kernels 4 and 5)");
        float* img = nullptr;
        if (!dev_alloc_t(s, &img, (size_t)N * D)) return fail(s, NG_ERR_OOM, "ring image");
        NG_CUDA(s, cudaMemsetAsync(img, 0, (size_t)N * D * 4, s->stream));
        NG_CUDA(s, cudaMemcpyAsync(img + (size_t)(n % D) * N, s->a.ring + (size_t)(n % 2) * N, (size_t)N * 4, cudaMemcpyDeviceToDevice, s->stream));
        if (s->queue_backend) materialize_queues_kernel<<<s->sm_count * 8, 256, 0, s->stream>>>(s->a, (long long)n, img);
        else materialize_window_kernel<<<s->sm_count * 8, 256, 0, s->stream>>>(s->a, (long long)n, img);
        NG_CUDA(s, cudaMemcpyAsync(user, img + first, (size_t)count * 4, cudaMemcpyDefault, s->stream));
        NG_CUDA(s, cudaStreamSynchronize(s->stream));
        dev_free(s, img);
        return NG_OK;
    }
    int64_t done = 0;
    while (done < count) {
        const int64_t e = first + done, slot = e / N, i0 = e % N;
        const int64_t len = std::min<int64_t>(count - done, N - i0);
        const int64_t np = n + (((slot - n) % D) + D) % D;               // the pending step stored in API slot `slot`
        float* dev = s->a.ring + (size_t)(np % Dr) * N + i0;
        char* usr = (char*)user + (size_t)done * 4;
        if (to_device) NG_CUDA(s, cudaMemcpyAsync(dev, usr, (size_t)len * 4, cudaMemcpyDefault, s->stream));
        else NG_CUDA(s, cudaMemcpyAsync(usr, dev, (size_t)len * 4, cudaMemcpyDefault, s->stream));
        done += len;
    }
    NG_CUDA(s, cudaStreamSynchronize(s->stream));
    return NG_OK;
}

}  // namespace

extern "C" {

int32_t ng_create(const ng_config* cfg, const ng_allocator* alloc, void* cuda_stream, ng_sim** out) {
    if (!out) return NG_ERR_INVALID_ARG;
    *out = nullptr;
    if (!cfg || !(cfg->dt_ms > 0.0) || cfg->ring_slots < 1 || cfg->ring_slots > 255 || cfg->max_recorded_spikes < 0)
        return NG_ERR_INVALID_ARG;
    if (cudaSetDevice(cfg->device) != cudaSuccess) { cudaGetLastError(); return NG_ERR_CUDA; }
    ng_sim* s = new ng_sim();
    s->cfg = *cfg;
    if (alloc && alloc->alloc && alloc->free) { s->alloc = *alloc; s->has_alloc = true; }
    if (cuda_stream) s->stream = (cudaStream_t)cuda_stream;
    else {
        if (cudaStreamCreateWithFlags(&s->stream, cudaStreamNonBlocking) != cudaSuccess) { delete s; return NG_ERR_CUDA; }
        s->own_stream = true;
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cfg->device) == cudaSuccess) {
        s->sm_count = prop.multiProcessorCount;
        s->l2_bytes = (size_t)prop.l2CacheSize;
        s->coop_ok = prop.cooperativeLaunch != 0;
    }
    *out = s;
    return NG_OK;
}

int32_t ng_destroy(ng_sim* s) {
    if (!s) return NG_OK;
    cudaSetDevice(s->cfg.device);
    if (s->stream) cudaStreamSynchronize(s->stream);
    destroy_graph(s);
    std::vector<void*> all = s->allocs;
    for (void* p : all) dev_free(s, p);
    for (int q = 0; q < 16; ++q) if (s->xchg_ipc_open[q] && s->a.xchg[q]) cudaIpcCloseMemHandle(s->a.xchg[q]);
    if (s->xchg_own) cudaFree(s->xchg_own);
    if (s->own_stream) cudaStreamDestroy(s->stream);
    delete s;
    return NG_OK;
}

const char* ng_last_error(const ng_sim* s) { return s ? s->err.c_str() : "null handle"; }

int32_t ng_create_population(ng_sim* s, int32_t n, const ng_lif_params* p, int32_t* first_id_out) {
    if (!s || !p) return NG_ERR_INVALID_ARG;
    if (s->prepared) return fail(s, NG_ERR_STATE, "population after ng_prepare");
    if (n <= 0 || (int64_t)s->N + n > 2147483000LL) return fail(s, NG_ERR_INVALID_ARG, "n <= 0 or too many neurons");
    if (s->pops.size() >= 255) return fail(s, NG_ERR_INVALID_ARG, "more than 255 populations");
    if (!(p->C_m > 0.0) || !(p->tau_m > 0.0) || !(p->tau_syn > 0.0) || p->t_ref_ms < 0.0 || p->poisson_rate_hz < 0.0)
        return fail(s, NG_ERR_INVALID_ARG, "non-positive C_m, tau_m or tau_syn, or negative t_ref / rate");
    if (std::fabs(p->tau_m - p->tau_syn) < 1e-9) return fail(s, NG_ERR_INVALID_ARG, "tau_m == tau_syn (DESIGN.md C19)");
    HostPop hp{};
    hp.first = s->N; hp.n = n; hp.p = *p;
    make_pop_dev(*p, s->cfg.dt_ms, hp.dev);
    if (!make_poisson_table(p->poisson_rate_hz * s->cfg.dt_ms * 1e-3, hp.dev))
        return fail(s, NG_ERR_INVALID_ARG, "Poisson rate * h too large for the 64-entry CDF table");
    s->pops.push_back(hp);
    s->N += n;
    if (first_id_out) *first_id_out = hp.first;
    return NG_OK;
}

int32_t ng_connect_fixed_indegree(ng_sim* s, int32_t src_first, int32_t src_n, int32_t tgt_first, int32_t tgt_n, int32_t K,
                                  const ng_dist* w, const ng_dist* d) {
    return add_call(s, kRuleIndegree, src_first, src_n, tgt_first, tgt_n, K, w, d);
}
int32_t ng_connect_fixed_outdegree(ng_sim* s, int32_t src_first, int32_t src_n, int32_t tgt_first, int32_t tgt_n, int32_t K,
                                   const ng_dist* w, const ng_dist* d) {
    return add_call(s, kRuleOutdegree, src_first, src_n, tgt_first, tgt_n, K, w, d);
}

int32_t ng_connect_fixed_indegree_port(ng_sim* s, int32_t src_first, int32_t src_n, int32_t tgt_first, int32_t tgt_n, int32_t K,
                                       const ng_dist* w, const ng_dist* d, int32_t port) {
    return add_call(s, kRuleIndegree, src_first, src_n, tgt_first, tgt_n, K, w, d, port);
}
int32_t ng_connect_fixed_outdegree_port(ng_sim* s, int32_t src_first, int32_t src_n, int32_t tgt_first, int32_t tgt_n, int32_t K,
                                        const ng_dist* w, const ng_dist* d, int32_t port) {
    return add_call(s, kRuleOutdegree, src_first, src_n, tgt_first, tgt_n, K, w, d, port);
}

int32_t ng_create_population_adex(ng_sim* s, int32_t n, const ng_adex_params* p, int32_t* first_id_out) {
    if (!s || !p) return NG_ERR_INVALID_ARG;
    if (s->prepared) return fail(s, NG_ERR_STATE, "population after ng_prepare");
    if (n <= 0 || (int64_t)s->N + n > 1073741000LL) return fail(s, NG_ERR_INVALID_ARG, "n <= 0 or too many neurons");
    if (s->pops.size() >= 255) return fail(s, NG_ERR_INVALID_ARG, "more than 255 populations");
    if (!(p->C_m > 0.0) || !(p->g_L > 0.0) || !(p->Delta_T > 0.0) || !(p->tau_w > 0.0) || !(p->tau_syn > 0.0) ||
        !(p->h_min > 0.0) || p->poisson_rate_hz < 0.0)
        return fail(s, NG_ERR_INVALID_ARG, "non-positive C_m, g_L, Delta_T, tau_w, tau_syn or h_min, or negative rate");
    for (int i = 0; i < 6; ++i) if (!(p->tol[i] > 0.0)) return fail(s, NG_ERR_INVALID_ARG, "non-positive tolerance");
    HostPop hp{};
    hp.first = s->N; hp.n = n;
    PopDev& d = hp.dev;
    d.model = 1;
    d.E_L = (float)p->E_L;                                 // initial V
    d.w_ext = (float)p->poisson_weight;
    AdexDev& x = d.ax;
    x.g_L = (float)p->g_L; x.E_L = (float)p->E_L; x.V_T = (float)p->V_T; x.inv_DeltaT = (float)(1.0 / p->Delta_T);
    x.gL_DeltaT = (float)(p->g_L * p->Delta_T); x.inv_C = (float)(1.0 / p->C_m); x.inv_tau_w = (float)(1.0 / p->tau_w);
    x.a = (float)p->a; x.b = (float)p->b; x.V_reset = (float)p->V_reset; x.V_peak = (float)p->V_peak;
    x.E_ex = (float)p->E_ex; x.E_in = (float)p->E_in; x.inv_tau_syn = (float)(1.0 / p->tau_syn); x.I_e = (float)p->I_e;
    x.jump = (float)(std::exp(1.0) / p->tau_syn);
    for (int i = 0; i < 6; ++i) x.inv_tol[i] = (float)(1.0 / p->tol[i]);
    x.h_min = (float)p->h_min;
    if (!make_poisson_table(p->poisson_rate_hz * s->cfg.dt_ms * 1e-3, d))
        return fail(s, NG_ERR_INVALID_ARG, "Poisson rate * h too large for the 64-entry CDF table");
    s->pops.push_back(hp);
    s->N += n;
    if (first_id_out) *first_id_out = hp.first;
    return NG_OK;
}

int32_t ng_shard_range(int32_t n_neurons, int32_t rank, int32_t world, int32_t* first_out, int32_t* n_out) {
    if (n_neurons < 0 || world < 1 || world > kMaxShards || rank < 0 || rank >= world || !first_out || !n_out) return NG_ERR_INVALID_ARG;
    const int32_t first = (int32_t)((int64_t)n_neurons * rank / world);
    *first_out = first;
    *n_out = (int32_t)((int64_t)n_neurons * (rank + 1) / world) - first;
    return NG_OK;
}

int32_t ng_set_shard(ng_sim* s, int32_t rank, int32_t world) {
    if (!s) return NG_ERR_INVALID_ARG;
    if (s->prepared) return fail(s, NG_ERR_STATE, "ng_set_shard after ng_prepare");
    if (world < 1 || world > kMaxShards || rank < 0 || rank >= world) return fail(s, NG_ERR_INVALID_ARG, "shard rank / world (1..16)");
    s->shard_rank = rank; s->shard_world = world;
    return NG_OK;
}

int32_t ng_exchange_handle(ng_sim* s, void* handle_out_64, void** local_ptr_out) {
    if (!s) return NG_ERR_INVALID_ARG;
    if (!s->prepared || s->shard_world < 2) return fail(s, NG_ERR_STATE, "no exchange buffer: ng_set_shard with world > 1, then ng_prepare");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    if (local_ptr_out) *local_ptr_out = s->xchg_own;
    if (handle_out_64) {
        static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handle size");
        cudaIpcMemHandle_t h;
        NG_CUDA(s, cudaIpcGetMemHandle(&h, s->xchg_own));
        std::memcpy(handle_out_64, &h, 64);
    }
    return NG_OK;
}

int32_t ng_exchange_attach(ng_sim* s, int32_t peer_rank, const void* ipc_handle_64, void* same_process_ptr) {
    if (!s) return NG_ERR_INVALID_ARG;
    if (!s->prepared || s->shard_world < 2) return fail(s, NG_ERR_STATE, "no exchange buffer: ng_set_shard with world > 1, then ng_prepare");
    if (peer_rank < 0 || peer_rank >= s->shard_world || peer_rank == s->shard_rank) return fail(s, NG_ERR_INVALID_ARG, "peer rank");
    if ((ipc_handle_64 == nullptr) == (same_process_ptr == nullptr)) return fail(s, NG_ERR_INVALID_ARG, "give the IPC handle or the pointer, not both");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    if (s->a.xchg[peer_rank]) return fail(s, NG_ERR_STATE, "peer already attached");
    if (ipc_handle_64) {
        cudaIpcMemHandle_t h;
        std::memcpy(&h, ipc_handle_64, 64);
        void* p = nullptr;
        NG_CUDA(s, cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess));
        s->a.xchg[peer_rank] = (unsigned char*)p; s->xchg_ipc_open[peer_rank] = true;
    } else {
        // a buffer of another handle in this process: on another device it needs peer access (NVLink / NVSwitch)
        cudaPointerAttributes at{};
        NG_CUDA(s, cudaPointerGetAttributes(&at, same_process_ptr));
        if (at.type != cudaMemoryTypeDevice) return fail(s, NG_ERR_INVALID_ARG, "not a device pointer");
        if (at.device != s->cfg.device) {
            cudaError_t e = cudaDeviceEnablePeerAccess(at.device, 0);
            if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) return fail(s, NG_ERR_CUDA, std::string("cudaDeviceEnablePeerAccess: ") + cudaGetErrorString(e));
            cudaGetLastError();
        }
        s->a.xchg[peer_rank] = (unsigned char*)same_process_ptr;
    }
    destroy_graph(s);                                              // the kernels' argument block changed
    return NG_OK;
}

int32_t ng_shard_phase(ng_sim* s, int32_t phase) {
    if (!s) return NG_ERR_INVALID_ARG;
    if (!s->prepared || s->shard_world < 2) return fail(s, NG_ERR_STATE, "ng_shard_phase needs a prepared target-sharded handle");
    if (phase != 0 && phase != 1) return fail(s, NG_ERR_INVALID_ARG, "phase is 0 (update + publish) or 1 (gather + deliver)");
    for (int q = 0; q < s->shard_world; ++q)
        if (!s->a.xchg[q]) return fail(s, NG_ERR_STATE, "target-sharded mode: ng_exchange_attach every peer first");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    if (phase == 0) { launch_update(s); launch_exchange_publish(s); s->launches_update += 1; }
    else { launch_exchange_gather(s); launch_deliver(s); s->launches_deliver += 1; s->steps_done += 1; }
    NG_CUDA(s, cudaGetLastError());
    return NG_OK;
}

int32_t ng_set_bypass(ng_sim* s, int32_t bypass, double fraction) {
    if (!s) return NG_ERR_INVALID_ARG;
    if (s->prepared) return fail(s, NG_ERR_STATE, "ng_set_bypass after ng_prepare");
    if (!(fraction >= 0.0) || fraction > 1.0) return fail(s, NG_ERR_INVALID_ARG, "fraction outside [0, 1]");
    s->bypass = bypass ? 1 : 0;
    double t = std::floor(fraction * 4294967296.0);
    if (t > 4294967295.0) t = 4294967295.0;
    s->inject_thr = (uint32_t)t;
    return NG_OK;
}

int32_t ng_set_option(ng_sim* s, int32_t option, int64_t value) {
    if (!s) return NG_ERR_INVALID_ARG;
    switch (option) {
        case NG_OPT_STEP_MODE:
            if (value < 0 || value > 3) return fail(s, NG_ERR_INVALID_ARG, "step mode is 0, 1, 2 or 3 (auto)");
            s->step_mode_opt = (int)value;
            if (s->prepared) configure_launch(s); else if (value != 3) s->step_mode = (int)value;
            break;
        case NG_OPT_STEPS_PER_GRAPH:
            if (value < 1 || value > 10000) return fail(s, NG_ERR_INVALID_ARG, "steps per graph in 1..10000");
            s->steps_per_graph = (int)value; destroy_graph(s); break;
        case NG_OPT_DELIVERY_KERNEL:
            if (value < 0 || value > 6) return fail(s, NG_ERR_INVALID_ARG, "delivery kernel is 0 .. 6");
            if (value == 6 && s->shard_world > 1) return fail(s, NG_ERR_INVALID_ARG, "delivery kernel 6 (pipelined) runs on one GPU only");
            if (value == 3 && s->shard_world > 1) return fail(s, NG_ERR_INVALID_ARG, "delivery kernel 3 (pipelined) runs on one GPU only");
            if (s->prepared && value != 0 && ((value == 4) != (s->window_backend && !s->pipewin) || (value == 5) != s->queue_backend || (value == 6) != s->pipewin))
                return fail(s, NG_ERR_STATE, "delivery kernels 4, 6 (spike-buffer backends) and 5 (event queues) must be chosen before ng_prepare and cannot be left after it");
            s->delivery_kernel_opt = (int)value; if (s->prepared) configure_launch(s); break;
        case NG_OPT_DELIVER_BLOCKS:
            if (value < 0 || value > (1 << 20)) return fail(s, NG_ERR_INVALID_ARG, "deliver blocks out of range");
            s->deliver_blocks_opt = (int)value; if (s->prepared) configure_launch(s); break;
        case NG_OPT_PROFILE: s->profile = value ? 1 : 0; break;
        case NG_OPT_ASYNC: s->async = value ? 1 : 0; break;
        case NG_OPT_SORT_SEGMENTS:
            if (s->prepared) return fail(s, NG_ERR_STATE, "NG_OPT_SORT_SEGMENTS after ng_prepare");
            s->sort_segments = value ? 1 : 0; break;
        case NG_OPT_TRACE:
            if (value && !s->prepared) return fail(s, NG_ERR_STATE, "NG_OPT_TRACE before ng_prepare");
            if (value && !s->a.trace && s->trace_saved) { s->a.trace = s->trace_saved; s->trace_saved = nullptr; }   // switched back on
            if (value && !s->a.trace) {
                const size_t words = (size_t)kTraceSteps * (size_t)s->sm_count * 32 * kTraceStamps;
                if (!dev_alloc_t(s, &s->a.trace, words)) return fail(s, NG_ERR_OOM, "trace buffer");
                NG_CUDA(s, cudaMemsetAsync(s->a.trace, 0, words * 8, s->stream));
                s->trace_on = true;
            }
            if (!value && s->a.trace) { s->trace_saved = s->a.trace; s->a.trace = nullptr; }
            break;
        case NG_OPT_PERSISTENT_THREADS:
            if (value != 512 && value != 1024) return fail(s, NG_ERR_INVALID_ARG, "persistent threads: 512 or 1024");
            s->persistent_threads = (int)value; if (s->prepared) configure_launch(s); break;
        case NG_OPT_PREFETCH: s->prefetch_opt = value ? 1 : 0; if (s->prepared) configure_launch(s); break;
        case NG_OPT_QUEUE_CAPACITY:
            if (s->prepared) return fail(s, NG_ERR_STATE, "NG_OPT_QUEUE_CAPACITY after ng_prepare");
            if (value < 0) return fail(s, NG_ERR_INVALID_ARG, "queue capacity < 0");
            s->queue_cap_opt = value; break;
        default: return fail(s, NG_ERR_INVALID_ARG, "unknown option");
    }
    return NG_OK;
}

int32_t ng_prepare(ng_sim* s) {
    if (!s) return NG_ERR_INVALID_ARG;
    if (s->prepared) return NG_OK;
    if (s->N <= 0) return fail(s, NG_ERR_STATE, "no population");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    const int N = s->N, D = s->cfg.ring_slots;               // N: neurons of the whole network = sources = rows
    // target-sharded mode: this handle owns the contiguous id range [id_first, id_first + NL) (ng_shard_range)
    s->id_first = (int32_t)((int64_t)N * s->shard_rank / s->shard_world);
    s->NL = (int32_t)((int64_t)N * (s->shard_rank + 1) / s->shard_world) - s->id_first;
    const int NL = s->NL;
    if (NL <= 0) return fail(s, NG_ERR_INVALID_ARG, "more shards than neurons");
    cudaStream_t st = s->stream;
    // Ring or spike window?  A ring that cannot stay in L2 (config 3: 65 planes x 4 MB) costs a DRAM round trip per plane
    // and step; the spike-buffer backend keeps two planes whatever D is and measured faster on every point of the
    // config 3 sweep, so it is the automatic choice there.
    s->S = 0;
    for (const CallDev& c : s->calls) s->S += (int64_t)(c.rule == kRuleIndegree ? c.tgt_n : c.src_n) * c.K;
    const int64_t S_all = s->S;
    s->S = S_all / s->shard_world;                              // estimate until the build has counted this shard's records
    s->has_adex = false;
    for (const HostPop& hp : s->pops) s->has_adex = s->has_adex || hp.dev.model == 1;
    s->NR = (int64_t)NL * (s->has_adex ? 2 : 1);
    const double ring_bytes = (double)s->NR * (D + 1) * 4.0;
    const bool beyond_l2 = (double)NL * (D + 1) * 4.0 > 0.8 * (double)s->l2_bytes;
    // Beyond L2, short delay groups (a few records per (source, delay): config 3 at out-degree 100 and 1000) make the
    // spike-buffer walk read at random 12-125-byte granularity; the event queues read a spiking row once, whole
    // (DESIGN.md section 7).  Expected events per step: the injected fraction in delivery-only mode, else 2 % of S.
    const double mean_group = (double)s->S / ((double)N * D);
    const double ev_step = s->bypass ? (double)s->inject_thr / 4294967296.0 * (double)s->S : 0.02 * (double)s->S;
    int64_t qcap = s->queue_cap_opt > 0 ? s->queue_cap_opt : (int64_t)(1.25 * ev_step) + 65536;
    qcap = (qcap + 1) & ~(int64_t)1;
    size_t mem_free = 0, mem_total = 0;
    cudaMemGetInfo(&mem_free, &mem_total);
    const bool queue_fits = (double)qcap * D * 8.0 + (double)s->S * 9.0 < 0.85 * (double)mem_total;
    // A ring of more than half the L2 does not stay resident next to the record stream (config 4: 84 MB; the two-port AdEx
    // network: 168 MB): the pipelined kernel then walks the spike window into two planes instead (kernel 6; config 4
    // 20.4 -> 17.7 us per step, AdEx 10^6 92.0 -> 88.5).  Latency-bound networks with a small ring keep kernel 3 (config 2:
    // 4.6 us against 10.0 with the window walk, which visits a spike once per delay group instead of once).
    s->pipewin = s->delivery_kernel_opt == 6 ||
                 (s->delivery_kernel_opt == 0 && s->step_mode_opt >= 2 && s->coop_ok && !s->bypass && D >= 2 && s->shard_world == 1 &&
                  ring_bytes > 0.5 * (double)s->l2_bytes && mean_group >= 16.0);
    if (s->pipewin && (!s->coop_ok || s->bypass || D < 2 || s->shard_world > 1))
        return fail(s, NG_ERR_INVALID_ARG, "delivery kernel 6 needs cooperative launch, a neuron update (no delivery-only mode), ring_slots >= 2 and one GPU");
    s->queue_backend = s->delivery_kernel_opt == 5 || (s->delivery_kernel_opt == 0 && beyond_l2 && mean_group < 48.0 && queue_fits && !s->pipewin);
    s->window_backend = s->pipewin || s->delivery_kernel_opt == 4 || (s->delivery_kernel_opt == 0 && beyond_l2 && !s->queue_backend);
    const int planes = (s->window_backend || s->queue_backend) ? 2 : D + 1;               // ring planes actually stored
    // Receptor port 1 is the inhibitory conductance of AdEx neurons: it exists only in networks with an AdEx population
    // (two-port ring planes), and only AdEx targets read it — a LIF target would silently drop such input.
    for (const CallDev& c : s->calls) {
        if (c.port != 1) continue;
        if (!s->has_adex) return fail(s, NG_ERR_INVALID_ARG, "receptor port 1 needs an AdEx population (LIF-only network has one port)");
        for (const HostPop& hp : s->pops)
            if (hp.dev.model != 1 && hp.first < c.tgt_first + c.tgt_n && c.tgt_first < hp.first + hp.n)
                return fail(s, NG_ERR_INVALID_ARG, "receptor port 1 onto a target range that holds LIF neurons (they have one port)");
    }
    const size_t NRs = (size_t)s->NR;

    cudaEvent_t e0, e1;
    NG_CUDA(s, cudaEventCreate(&e0));
    NG_CUDA(s, cudaEventCreate(&e1));
    NG_CUDA(s, cudaEventRecord(e0, st));

    // ---- control block, populations, state ----
    // the spike array of two steps; of four where the resident LIF kernel with the split barrier can be chosen (its CTAs
    // drift a phase apart; one neuron per updater thread of a persistent launch: small networks, 80 B per neuron)
    s->list_bufs = (!s->has_adex && s->shard_world <= 1 && (long long)N <= 1024LL * 4 * std::max(1, s->sm_count)) ? 4 : 2;
    bool ok = dev_alloc_t(s, &s->d_ctl, 1) && dev_alloc_t(s, &s->d_pops, s->pops.size()) &&
              dev_alloc_t(s, &s->d_pop_of, (size_t)NL) && dev_alloc_t(s, &s->a.V, (size_t)NL) &&
              dev_alloc_t(s, &s->a.I, (size_t)NL) && dev_alloc_t(s, &s->a.refr, (size_t)NL) &&
              dev_alloc_t(s, &s->a.ring, NRs * planes) && dev_alloc_t(s, &s->a.spike_list, (size_t)s->list_bufs * N) &&
              dev_alloc_t(s, &s->a.spike_row, (size_t)s->list_bufs * N) && dev_alloc_t(s, &s->a.pois_k, (size_t)NL) && dev_alloc_t(s, &s->d_row_info, (size_t)N) &&
              dev_alloc_t(s, &s->d_calls, std::max<size_t>(1, s->calls.size())) &&
              dev_alloc_t(s, &s->d_cnt, (size_t)N * D) && dev_alloc_t(s, &s->d_row_len, (size_t)N) &&
              dev_alloc_t(s, &s->d_row_off, (size_t)N + 1) && dev_alloc_t(s, &s->d_grp_rel, (size_t)N * (D + 1));
    if (ok && (s->cfg.flags & NG_DEBUG_INPUT)) ok = dev_alloc_t(s, &s->a.last_input, NRs);
    if (ok && s->has_adex)
        ok = dev_alloc_t(s, &s->a.ax_w, (size_t)NL) && dev_alloc_t(s, &s->a.ax_gx, (size_t)NL) && dev_alloc_t(s, &s->a.ax_yx, (size_t)NL) &&
             dev_alloc_t(s, &s->a.ax_gi, (size_t)NL) && dev_alloc_t(s, &s->a.ax_yi, (size_t)NL) && dev_alloc_t(s, &s->a.ax_h, (size_t)NL);
    if (ok && (s->cfg.flags & NG_RECORD_SPIKES) && s->cfg.max_recorded_spikes > 0) {
        ok = dev_alloc_t(s, &s->a.rec_step, (size_t)s->cfg.max_recorded_spikes) &&
             dev_alloc_t(s, &s->a.rec_id, (size_t)s->cfg.max_recorded_spikes);
        s->a.rec_cap = s->cfg.max_recorded_spikes;
    }
    if (!ok) return fail(s, NG_ERR_OOM, "device allocation failed (state)");
    NG_CUDA(s, cudaMemsetAsync(s->d_ctl, 0, sizeof(Ctl), st));
    NG_CUDA(s, cudaMemsetAsync(s->a.I, 0, (size_t)NL * 4, st));
    NG_CUDA(s, cudaMemsetAsync(s->a.refr, 0, (size_t)NL * 4, st));
    NG_CUDA(s, cudaMemsetAsync(s->a.ring, 0, NRs * planes * 4, st));
    if (s->has_adex) {
        for (float* p : {s->a.ax_w, s->a.ax_gx, s->a.ax_yx, s->a.ax_gi, s->a.ax_yi}) NG_CUDA(s, cudaMemsetAsync(p, 0, (size_t)NL * 4, st));
        std::vector<float> h0((size_t)NL, (float)s->cfg.dt_ms);    // sub-step size starts at the whole time step
        NG_CUDA(s, cudaMemcpyAsync(s->a.ax_h, h0.data(), (size_t)NL * 4, cudaMemcpyHostToDevice, st));
        NG_CUDA(s, cudaStreamSynchronize(st));
    }
    if (s->window_backend) {
        // worst case N spikes per step for D steps; beyond 2^26 entries an eighth of that (overflow is detected)
        const long long worst = (long long)N * D;
        s->a.win_cap = worst <= (1LL << 26) ? worst : std::max(1LL << 26, worst / 8);
        if (!dev_alloc_t(s, &s->a.win_id, (size_t)s->a.win_cap)) return fail(s, NG_ERR_OOM, "device allocation failed (spike window)");
    }
    if (s->queue_backend) {
        s->a.q_cap = qcap;
        if (!(dev_alloc_t(s, &s->a.q_ev, (size_t)qcap * D) && dev_alloc_t(s, &s->a.q_tail, (size_t)D * kQTailStride)))
            return fail(s, NG_ERR_OOM, "device allocation failed (event queues)");
        NG_CUDA(s, cudaMemsetAsync(s->a.q_tail, 0, (size_t)D * kQTailStride * 8, st));
    }
    NG_CUDA(s, cudaMemsetAsync(s->d_cnt, 0, (size_t)N * D * 4, st));
    if (s->a.last_input) NG_CUDA(s, cudaMemsetAsync(s->a.last_input, 0, NRs * 4, st));
    std::vector<PopDev> pd(s->pops.size());
    for (size_t i = 0; i < s->pops.size(); ++i) pd[i] = s->pops[i].dev;
    NG_CUDA(s, cudaMemcpyAsync(s->d_pops, pd.data(), pd.size() * sizeof(PopDev), cudaMemcpyHostToDevice, st));
    if (!s->calls.empty())
        NG_CUDA(s, cudaMemcpyAsync(s->d_calls, s->calls.data(), s->calls.size() * sizeof(CallDev), cudaMemcpyHostToDevice, st));
    for (size_t i = 0; i < s->pops.size(); ++i) {                  // the part of each population this shard owns
        const HostPop& hp = s->pops[i];
        const int lo = std::max(hp.first, s->id_first), hi = std::min(hp.first + hp.n, s->id_first + NL);
        if (hi <= lo) continue;
        fill_pop_of_kernel<<<(hi - lo + 255) / 256, 256, 0, st>>>(s->d_pop_of, s->a.V, lo - s->id_first, hi - lo, (uint8_t)i, hp.dev.E_L);
        s->launches_other++;
    }
    if (s->shard_world > 1) {
        // receive buffer of the per-step spike exchange: plain cudaMalloc (it is exported to the peers as a CUDA IPC
        // handle, which the pooled allocations of the caller's allocator cannot be)
        s->a.xchg_cap = (int32_t)(((int64_t)N + s->shard_world - 1) / s->shard_world + 1);
        s->xchg_bytes = (size_t)kXchgHeaderBytes + (size_t)2 * s->shard_world * (size_t)s->a.xchg_cap * 4;
        if (cudaMalloc((void**)&s->xchg_own, s->xchg_bytes) != cudaSuccess) { cudaGetLastError(); return fail(s, NG_ERR_OOM, "device allocation failed (exchange buffer)"); }
        NG_CUDA(s, cudaMemsetAsync(s->xchg_own, 0, s->xchg_bytes, st));
        s->a.xchg[s->shard_rank] = s->xchg_own;
        s->a.xchg_rank = s->shard_rank; s->a.xchg_world = s->shard_world;
    }

    // ---- connection build (a0) ----
    const uint32_t seed_lo = (uint32_t)s->cfg.seed, seed_hi = (uint32_t)(s->cfg.seed >> 32);
    const int cap = s->sm_count * 16;
    // draws the build kernels of this shard regenerate for one call: fixed in-degree -> the local targets only
    auto call_draws = [&](const CallDev& c) -> long long {
        if (c.rule != kRuleIndegree) return (long long)c.src_n * c.K;
        const int lo = std::max(c.tgt_first, s->id_first), hi = std::min(c.tgt_first + c.tgt_n, s->id_first + NL);
        return (long long)std::max(0, hi - lo) * c.K;
    };
    for (size_t ci = 0; ci < s->calls.size(); ++ci) {
        const CallDev& c = s->calls[ci];
        const long long total = call_draws(c);
        if (total == 0) continue;
        build_count_kernel<<<grid_for(total, 256, cap), 256, 0, st>>>(s->d_calls, (int)ci, seed_lo, seed_hi, D, s->d_cnt, s->d_ctl, s->id_first, NL);
        s->launches_other++;
    }
    build_rowlen_kernel<<<(N + 255) / 256, 256, 0, st>>>(s->d_cnt, N, D, s->d_row_len, s->d_ctl);
    scan_exclusive_kernel<<<1, 1024, 0, st>>>(s->d_row_len, s->d_row_off, N, s->d_ctl);
    build_groups_kernel<<<(N + 255) / 256, 256, 0, st>>>(s->d_cnt, N, D, s->d_grp_rel);
    build_row_info_kernel<<<(N + 255) / 256, 256, 0, st>>>(N, D, s->d_row_off, s->d_grp_rel, s->d_row_info);
    s->launches_other += 4;
    Ctl h{};
    int32_t rc = read_ctl(s, &h);
    if (rc) return rc;
    NG_CUDA(s, cudaGetLastError());
    if (h.err_delay) return fail(s, NG_ERR_OVERFLOW, "a drawn delay fell outside [1, ring_slots]");
    s->n_padded = (int64_t)h.n_padded;
    s->max_row_records = h.max_row_records;
    s->S = (int64_t)h.n_records;                                    // connections stored on this shard (= all of them on one GPU)
    if (s->shard_world == 1 && s->S != S_all) return fail(s, NG_ERR_CUDA, "builder lost records");
    const size_t np = (size_t)std::max<int64_t>(s->n_padded, 4);
    if (!(dev_alloc_t(s, &s->d_tgt, np) && dev_alloc_t(s, &s->d_w, np) && dev_alloc_t(s, &s->d_dly, np + 16)))
        return fail(s, NG_ERR_OOM, "device allocation failed (connection records)");
    NG_CUDA(s, cudaMemsetAsync(s->d_tgt, 0xFF, np * 4, st));       // padding records: target -1, weight 0, delay 0
    NG_CUDA(s, cudaMemsetAsync(s->d_w, 0, np * 4, st));
    NG_CUDA(s, cudaMemsetAsync(s->d_dly, 0, np, st));
    for (size_t ci = 0; ci < s->calls.size(); ++ci) {
        const CallDev& c = s->calls[ci];
        const long long total = call_draws(c);
        if (total == 0) continue;
        build_fill_kernel<<<grid_for(total, 256, cap), 256, 0, st>>>(s->d_calls, (int)ci, seed_lo, seed_hi, D, s->d_cnt,
                                                                   s->d_row_off, s->d_grp_rel, s->d_tgt, s->d_w, s->d_dly, NL, s->id_first);
        s->launches_other++;
    }
    long long* d_long = nullptr;
    if (s->sort_segments) {
        // groups beyond the warp sort's shared-memory tile go to a list; there are at most S / kSortMax of them
        const uint32_t long_cap = (uint32_t)std::min<int64_t>(s->S / kSortMax + 1, 0x7fffffff);
        if (!dev_alloc_t(s, &d_long, (size_t)long_cap)) return fail(s, NG_ERR_OOM, "device allocation failed (long-group list)");
        build_sort_groups_kernel<<<s->sm_count * 8, 256, 0, st>>>(N, D, s->d_row_off, s->d_grp_rel, s->d_tgt, s->d_w, d_long, long_cap, s->d_ctl);
        build_sort_long_groups_kernel<<<s->sm_count * 2, 1024, 0, st>>>(D, s->d_row_off, s->d_grp_rel, s->d_tgt, s->d_w, d_long, long_cap, s->d_ctl);
        s->launches_other += 2;
    }
    NG_CUDA(s, cudaEventRecord(e1, st));
    NG_CUDA(s, cudaStreamSynchronize(st));
    NG_CUDA(s, cudaGetLastError());
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    s->build_ms = ms;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    // the per-(source, delay) counters and the row lengths are builder scratch
    dev_free(s, s->d_cnt); s->d_cnt = nullptr;
    dev_free(s, s->d_row_len); s->d_row_len = nullptr;
    dev_free(s, d_long);

    // ---- step arguments ----
    s->a.NR = (int32_t)s->NR; s->a.dt_ms = (float)s->cfg.dt_ms; s->a.has_adex = s->has_adex ? 1 : 0;
    s->a.N = NL; s->a.NS = N; s->a.id_first = s->id_first; s->a.D = D; s->a.Dr = planes; s->a.n_pops = (int32_t)s->pops.size(); s->a.seed_lo = seed_lo; s->a.seed_hi = seed_hi;
    s->a.pop_of = s->d_pop_of; s->a.pops = s->d_pops;
    s->a.row_info = s->d_row_info;
    s->a.row_off = s->d_row_off; s->a.grp_rel = s->d_grp_rel; s->a.tgt = s->d_tgt; s->a.w = s->d_w; s->a.dly = s->d_dly;
    s->a.ctl = s->d_ctl; s->a.bypass = s->bypass; s->a.inject_thr = s->inject_thr;
    s->prepared = true;
    configure_launch(s);
    return NG_OK;
}

int32_t ng_set_state(ng_sim* s, int32_t field, const void* data, int64_t count, int64_t first) {
    if (!s || !data) return NG_ERR_INVALID_ARG;
    if (!s->prepared) return fail(s, NG_ERR_STATE, "ng_set_state before ng_prepare");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    if (field == NG_FIELD_STEP) {
        if (count != 1 || first != 0) return fail(s, NG_ERR_INVALID_ARG, "NG_FIELD_STEP is one int64");
        long long n = 0;
        NG_CUDA(s, cudaMemcpy(&n, data, 8, cudaMemcpyDefault));
        if (n < 0) return fail(s, NG_ERR_INVALID_ARG, "negative step");
        Ctl h{};
        int32_t rc = read_ctl(s, &h);
        if (rc) return rc;
        const unsigned long long recorded = h.rec_total[h.step_u & 1];
        h.step_u = n; h.step_d = n; h.spike_cnt[0] = h.spike_cnt[1] = h.spike_cnt[2] = h.spike_cnt[3] = 0; h.ticket = 0; h.pending = 0;
        std::memset(h.win_start, 0, sizeof(h.win_start)); h.err_window = 0; h.win_tail = 0;
        h.slot = (int32_t)(n % s->a.Dr);
        h.rec_total[0] = h.rec_total[1] = recorded;
        h.err_queue = 0;
        NG_CUDA(s, cudaMemcpyAsync(s->d_ctl, &h, sizeof(Ctl), cudaMemcpyHostToDevice, s->stream));
        if (s->a.q_tail) NG_CUDA(s, cudaMemsetAsync(s->a.q_tail, 0, (size_t)s->cfg.ring_slots * kQTailStride * 8, s->stream));
        // target-sharded mode: forget the step stamps of the exchange (every rank must set the same step while all are idle)
        if (s->xchg_own) NG_CUDA(s, cudaMemsetAsync(s->xchg_own, 0, kXchgHeaderBytes, s->stream));
        NG_CUDA(s, cudaStreamSynchronize(s->stream));
        return NG_OK;
    }
    if (field == NG_FIELD_LAST_INPUT) return fail(s, NG_ERR_INVALID_ARG, "NG_FIELD_LAST_INPUT is read-only");
    void* base; size_t elem; int64_t len;
    int32_t rc = field_info(s, field, &base, &elem, &len);
    if (rc) return rc;
    if (count < 0 || first < 0 || first + count > len) return fail(s, NG_ERR_INVALID_ARG, "range outside the field");
    if (field == NG_FIELD_RING) return ring_copy(s, true, const_cast<void*>(data), count, first);
    NG_CUDA(s, cudaMemcpyAsync((char*)base + first * elem, data, (size_t)count * elem, cudaMemcpyDefault, s->stream));
    NG_CUDA(s, cudaStreamSynchronize(s->stream));
    return NG_OK;
}

int32_t ng_get_state(ng_sim* s, int32_t field, void* out, int64_t count, int64_t first) {
    if (!s || !out) return NG_ERR_INVALID_ARG;
    if (!s->prepared) return fail(s, NG_ERR_STATE, "ng_get_state before ng_prepare");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    if (field == NG_FIELD_STEP) {
        if (count != 1 || first != 0) return fail(s, NG_ERR_INVALID_ARG, "NG_FIELD_STEP is one int64");
        Ctl h{};
        int32_t rc = read_ctl(s, &h);
        if (rc) return rc;
        long long n = h.step_u;
        NG_CUDA(s, cudaMemcpy(out, &n, 8, cudaMemcpyDefault));
        return NG_OK;
    }
    void* base; size_t elem; int64_t len;
    int32_t rc = field_info(s, field, &base, &elem, &len);
    if (rc) return rc;
    if (count < 0 || first < 0 || first + count > len) return fail(s, NG_ERR_INVALID_ARG, "range outside the field");
    if (field == NG_FIELD_RING) return ring_copy(s, false, out, count, first);
    NG_CUDA(s, cudaMemcpyAsync(out, (char*)base + first * elem, (size_t)count * elem, cudaMemcpyDefault, s->stream));
    NG_CUDA(s, cudaStreamSynchronize(s->stream));
    return NG_OK;
}

int32_t ng_simulate(ng_sim* s, int64_t n_steps) {
    if (!s) return NG_ERR_INVALID_ARG;
    if (n_steps < 0) return fail(s, NG_ERR_INVALID_ARG, "n_steps < 0");
    int32_t rc = ng_prepare(s);
    if (rc) return rc;
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    if (n_steps == 0) return NG_OK;
    if (s->shard_world > 1)
        for (int q = 0; q < s->shard_world; ++q)
            if (!s->a.xchg[q]) return fail(s, NG_ERR_STATE, "target-sharded mode: ng_exchange_attach every peer before ng_simulate");
    cudaStream_t st = s->stream;
    if (s->profile && s->delivery_kernel != 6) {
        // per-kernel device times: events around every launch, read back in batches
        const int kBatch = 128;
        std::vector<cudaEvent_t> ev(3 * kBatch);
        for (auto& e : ev) NG_CUDA(s, cudaEventCreate(&e));
        for (int64_t done = 0; done < n_steps;) {
            const int b = (int)std::min<int64_t>(kBatch, n_steps - done);
            for (int i = 0; i < b; ++i) {
                cudaEventRecord(ev[3 * i], st);
                if (s->delivery_kernel == 3) launch_pipe(s); else launch_update(s);
                if (s->shard_world > 1) { launch_exchange_publish(s); launch_exchange_gather(s); }
                cudaEventRecord(ev[3 * i + 1], st);
                if (s->delivery_kernel != 3) launch_deliver(s);
                cudaEventRecord(ev[3 * i + 2], st);
            }
            NG_CUDA(s, cudaStreamSynchronize(st));
            for (int i = 0; i < b; ++i) {
                float m0 = 0, m1 = 0;
                cudaEventElapsedTime(&m0, ev[3 * i], ev[3 * i + 1]);
                cudaEventElapsedTime(&m1, ev[3 * i + 1], ev[3 * i + 2]);
                s->ms_update += m0; s->ms_deliver += m1;
            }
            done += b;
        }
        for (auto& e : ev) cudaEventDestroy(e);
        s->launches_update += n_steps; s->launches_deliver += s->delivery_kernel == 3 ? 0 : n_steps;
    } else if (s->step_mode == 2) {
        long long ns = n_steps;
        void* args[] = {(void*)&s->a, (void*)&ns};
        NG_CUDA(s, cudaMemsetAsync(&s->d_ctl->bar, 0, offsetof(Ctl, bar_list) + 2 * sizeof(BarWord) - offsetof(Ctl, bar), st));   // bar, ticket, bar_plane, bar_list
        const bool piped = s->delivery_kernel == 3 || s->delivery_kernel == 6;
        s->last_persistent_blocks = piped ? s->persistent_pipe_blocks : s->persistent_blocks;
        s->step_kernel = 0;
        if (s->delivery_kernel == 6) {
            s->step_kernel = 1;
            const void* fn = s->has_adex ? (s->one_round_persistent ? (const void*)persistent_pipe_kernel<true, true, false, true>
                                                                     : (const void*)persistent_pipe_kernel<true, false, false, true>)
                                         : (s->one_round_persistent && !s->bypass ? (const void*)persistent_pipe_kernel<false, true, false, true>
                                            : s->resm_bytes ? (const void*)persistent_pipe_kernel<false, false, true, true>
                                                            : (const void*)persistent_pipe_kernel<false, false, false, true>);
            NG_CUDA(s, cudaLaunchCooperativeKernel(fn, dim3(s->persistent_pipe_blocks),
                                                   dim3(s->has_adex ? 512 : s->persistent_threads), args,
                                                   s->has_adex || s->one_round_persistent ? 0 : s->resm_bytes, st));
        } else if (s->delivery_kernel == 3) {
            s->step_kernel = s->has_adex || !(s->one_round_persistent && !s->bypass) || !early_decision(s) ? 1 : NG_SPLIT_KERNEL ? 3 : 2;
            const void* fn = s->has_adex ? (s->one_round_persistent ? (const void*)persistent_pipe_kernel<true, true>
                                                                     : (const void*)persistent_pipe_kernel<true, false>)
                                         : (s->one_round_persistent && !s->bypass
                                                ? (early_decision(s) ? (NG_SPLIT_KERNEL ? (const void*)persistent_split_kernel : (const void*)persistent_pipe_kernel<false, true, false, false, true>)
                                                                     : (const void*)persistent_pipe_kernel<false, true>)
                                            : s->resm_bytes ? (const void*)persistent_pipe_kernel<false, false, true>
                                                            : (const void*)persistent_pipe_kernel<false, false>);
            NG_CUDA(s, cudaLaunchCooperativeKernel(fn, dim3(s->persistent_pipe_blocks),
                                                   dim3(s->has_adex ? 512 : s->persistent_threads), args,
                                                   s->has_adex || s->one_round_persistent ? 0 : s->resm_bytes, st));
        } else {
            const void* fn = s->delivery_kernel == 4 ? (const void*)persistent_kernel<4>
                             : s->delivery_kernel == 2 ? (const void*)persistent_kernel<2> : (const void*)persistent_kernel<1>;
            NG_CUDA(s, cudaLaunchCooperativeKernel(fn, dim3(s->persistent_blocks), dim3(s->persistent_threads), args, 0, st));
        }
        s->launches_update += 1;
    } else if (s->step_mode == 1) {
        for (int64_t i = 0; i < n_steps; ++i) launch_step(s);
        s->launches_update += n_steps; s->launches_deliver += s->delivery_kernel == 3 ? 0 : n_steps;
    } else {
        int64_t left = n_steps;
        const int G = s->steps_per_graph;
        if (left >= G) {
            if (!s->graph_exec || s->graph_steps != G) { rc = build_graph(s, G); if (rc) return rc; }
            while (left >= G) { NG_CUDA(s, cudaGraphLaunch(s->graph_exec, st)); left -= G; }
        }
        for (int64_t i = 0; i < left; ++i) launch_step(s);
        s->launches_update += n_steps; s->launches_deliver += s->delivery_kernel == 3 ? 0 : n_steps;
    }
    if (s->delivery_kernel == 3 && (s->profile || s->step_mode != 2)) { launch_pipe_flush(s); s->launches_deliver += 1; }
    NG_CUDA(s, cudaGetLastError());
    s->steps_done += (uint64_t)n_steps;
    if (s->async) return NG_OK;
    NG_CUDA(s, cudaStreamSynchronize(st));
    if (s->a.rec_cap > 0 || s->window_backend || s->queue_backend || s->shard_world > 1) {
        Ctl h{};
        rc = read_ctl(s, &h);
        if (rc) return rc;
        if (h.err_xchg) return fail(s, NG_ERR_CUDA, "spike exchange: a peer's spike list did not arrive within the bounded wait");
        if (h.err_window) return fail(s, NG_ERR_OVERFLOW, "spike window overflowed: more spikes within ring_slots steps than its capacity");
        if (h.err_queue) return fail(s, NG_ERR_OVERFLOW, "an event queue overflowed (events were dropped): raise NG_OPT_QUEUE_CAPACITY");
        const unsigned long long total = h.rec_total[h.step_u & 1];
        if (s->a.rec_cap > 0 && total > (unsigned long long)s->a.rec_cap) return fail(s, NG_ERR_OVERFLOW, "spike record full; later spikes were not recorded");
    }
    return NG_OK;
}

int32_t ng_get_spikes(ng_sim* s, int32_t* steps_host, int32_t* ids_host, int64_t capacity, int64_t* count_out) {
    if (!s || !count_out || capacity < 0) return NG_ERR_INVALID_ARG;
    *count_out = 0;
    if (!s->prepared) return fail(s, NG_ERR_STATE, "ng_get_spikes before ng_prepare");
    if (s->a.rec_cap <= 0) return fail(s, NG_ERR_STATE, "spike recording is not enabled (NG_RECORD_SPIKES)");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    Ctl h{};
    int32_t rc = read_ctl(s, &h);
    if (rc) return rc;
    const unsigned long long total = h.rec_total[h.step_u & 1];
    const int64_t have = (int64_t)std::min<unsigned long long>(total, (unsigned long long)s->a.rec_cap);
    if (total > (unsigned long long)s->a.rec_cap) s->rec_dropped += total - (unsigned long long)s->a.rec_cap;
    *count_out = have;
    const int64_t m = std::min(have, capacity);
    if (m == 0 || !steps_host || !ids_host) {
        if (total > (unsigned long long)s->a.rec_cap) {       // forget the uncounted tail so it is not double-counted
            h.rec_total[0] = h.rec_total[1] = (unsigned long long)have;
            NG_CUDA(s, cudaMemcpy(s->d_ctl, &h, sizeof(Ctl), cudaMemcpyHostToDevice));
        }
        return NG_OK;
    }
    NG_CUDA(s, cudaMemcpy(steps_host, s->a.rec_step, (size_t)m * 4, cudaMemcpyDeviceToHost));
    NG_CUDA(s, cudaMemcpy(ids_host, s->a.rec_id, (size_t)m * 4, cudaMemcpyDeviceToHost));
    const int64_t rest = have - m;
    if (rest > 0) {                                           // partial drain: move the tail to the front via scratch
        int32_t* tmp = nullptr;
        if (!dev_alloc_t(s, &tmp, (size_t)rest)) return fail(s, NG_ERR_OOM, "scratch for partial drain");
        NG_CUDA(s, cudaMemcpy(tmp, s->a.rec_step + m, (size_t)rest * 4, cudaMemcpyDeviceToDevice));
        NG_CUDA(s, cudaMemcpy(s->a.rec_step, tmp, (size_t)rest * 4, cudaMemcpyDeviceToDevice));
        NG_CUDA(s, cudaMemcpy(tmp, s->a.rec_id + m, (size_t)rest * 4, cudaMemcpyDeviceToDevice));
        NG_CUDA(s, cudaMemcpy(s->a.rec_id, tmp, (size_t)rest * 4, cudaMemcpyDeviceToDevice));
        dev_free(s, tmp);
    }
    h.rec_total[0] = h.rec_total[1] = (unsigned long long)rest;
    NG_CUDA(s, cudaMemcpy(s->d_ctl, &h, sizeof(Ctl), cudaMemcpyHostToDevice));
    return NG_OK;
}

int32_t ng_get_last_spikes(ng_sim* s, int32_t* ids_host, int64_t capacity, int64_t* count_out) {
    if (!s || !count_out || capacity < 0) return NG_ERR_INVALID_ARG;
    *count_out = 0;
    if (!s->prepared) return fail(s, NG_ERR_STATE, "ng_get_last_spikes before ng_prepare");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    Ctl h{};
    int32_t rc = read_ctl(s, &h);
    if (rc) return rc;
    if (h.step_u == 0) return NG_OK;
    const long long n = h.step_u - 1;
    // spike_cnt[n&3] is cleared only during step n+3 at the earliest; after step n it still holds step n's count
    const int64_t M = h.spike_cnt[n & 3];
    *count_out = M;
    const int64_t m = std::min(M, capacity);
    if (m > 0 && ids_host)
        NG_CUDA(s, cudaMemcpy(ids_host, s->a.spike_list + (size_t)(n & 1) * s->N, (size_t)m * 4, cudaMemcpyDeviceToHost));
    return NG_OK;
}

int32_t ng_copy_row_offsets(ng_sim* s, int64_t* out) {
    if (!s || !out) return NG_ERR_INVALID_ARG;
    if (!s->prepared) return fail(s, NG_ERR_STATE, "before ng_prepare");
    NG_CUDA(s, cudaMemcpy(out, s->d_row_off, ((size_t)s->N + 1) * 8, cudaMemcpyDefault));
    return NG_OK;
}
int32_t ng_copy_group_offsets(ng_sim* s, uint32_t* out) {
    if (!s || !out) return NG_ERR_INVALID_ARG;
    if (!s->prepared) return fail(s, NG_ERR_STATE, "before ng_prepare");
    NG_CUDA(s, cudaMemcpy(out, s->d_grp_rel, (size_t)s->N * (s->cfg.ring_slots + 1) * 4, cudaMemcpyDefault));
    return NG_OK;
}
int32_t ng_copy_records(ng_sim* s, int64_t first, int64_t count, int32_t* tgt, float* w, uint8_t* delay) {
    if (!s) return NG_ERR_INVALID_ARG;
    if (!s->prepared) return fail(s, NG_ERR_STATE, "before ng_prepare");
    if (first < 0 || count < 0 || first + count > s->n_padded) return fail(s, NG_ERR_INVALID_ARG, "record range");
    if (count == 0) return NG_OK;
    if (tgt) NG_CUDA(s, cudaMemcpy(tgt, s->d_tgt + first, (size_t)count * 4, cudaMemcpyDefault));
    if (w) NG_CUDA(s, cudaMemcpy(w, s->d_w + first, (size_t)count * 4, cudaMemcpyDefault));
    if (delay) NG_CUDA(s, cudaMemcpy(delay, s->d_dly + first, (size_t)count, cudaMemcpyDefault));
    return NG_OK;
}

int32_t ng_get_connections(ng_sim* s, int32_t src_id, int32_t* tgt_host, float* w_host, uint8_t* delay_host, int64_t capacity,
                           int64_t* count_out) {
    if (!s || !count_out || capacity < 0) return NG_ERR_INVALID_ARG;
    *count_out = 0;
    if (!s->prepared) return fail(s, NG_ERR_STATE, "before ng_prepare");
    if (src_id < 0 || src_id >= s->N) return fail(s, NG_ERR_INVALID_ARG, "source id");
    long long off = 0; uint32_t deg = 0;
    NG_CUDA(s, cudaMemcpy(&off, s->d_row_off + src_id, 8, cudaMemcpyDeviceToHost));
    NG_CUDA(s, cudaMemcpy(&deg, s->d_grp_rel + (size_t)src_id * (s->cfg.ring_slots + 1) + s->cfg.ring_slots, 4, cudaMemcpyDeviceToHost));
    *count_out = deg;
    const int64_t m = std::min<int64_t>(deg, capacity);
    if (m == 0) return NG_OK;
    if (tgt_host) NG_CUDA(s, cudaMemcpy(tgt_host, s->d_tgt + off, (size_t)m * 4, cudaMemcpyDeviceToHost));
    if (w_host) NG_CUDA(s, cudaMemcpy(w_host, s->d_w + off, (size_t)m * 4, cudaMemcpyDeviceToHost));
    if (delay_host) NG_CUDA(s, cudaMemcpy(delay_host, s->d_dly + off, (size_t)m, cudaMemcpyDeviceToHost));
    return NG_OK;
}

int32_t ng_get_stats(ng_sim* s, ng_stats* out) {
    if (!s || !out) return NG_ERR_INVALID_ARG;
    std::memset(out, 0, sizeof(*out));
    out->n_neurons = s->prepared ? s->NL : s->N;
    out->n_sources = s->N; out->shard_rank = s->shard_rank; out->shard_world = s->shard_world; out->id_first = s->id_first; out->step_kernel = s->step_kernel;
    out->step_mode = s->step_mode;
    if (!s->prepared) return NG_OK;
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    Ctl h{};
    int32_t rc = read_ctl(s, &h);
    if (rc) return rc;
    out->steps = s->steps_done; out->spikes = h.spikes; out->events = h.events;
    const unsigned long long total = h.rec_total[h.step_u & 1];
    out->recorded_dropped = s->rec_dropped + (s->a.rec_cap > 0 && total > (unsigned long long)s->a.rec_cap ? total - s->a.rec_cap : 0);
    out->n_connections = s->S; out->n_records_padded = s->n_padded; out->max_row_records = s->max_row_records;
    out->build_ms = s->build_ms; out->ms_update = s->ms_update; out->ms_deliver = s->ms_deliver;
    out->launches_update = s->launches_update; out->launches_deliver = s->launches_deliver; out->launches_other = s->launches_other;
    out->delivery_kernel = s->delivery_kernel;
    return NG_OK;
}

int32_t ng_enable_statistics(ng_sim* s, int64_t start_step, int32_t bin_steps, int32_t sample_per_pop, int32_t max_bins) {
    if (!s) return NG_ERR_INVALID_ARG;
    if (!s->prepared) return fail(s, NG_ERR_STATE, "ng_enable_statistics before ng_prepare");
    if (s->a.st_cnt) return fail(s, NG_ERR_STATE, "statistics are already enabled");
    if (s->shard_world > 1) return fail(s, NG_ERR_STATE, "on-device statistics are not available in target-sharded mode");
    if (start_step < 0 || bin_steps < 1 || sample_per_pop < 0 || max_bins < 1 || max_bins > (1 << 24))
        return fail(s, NG_ERR_INVALID_ARG, "start_step < 0, bin_steps < 1, sample_per_pop < 0 or max_bins outside 1..2^24");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    const size_t N = (size_t)s->N;
    // the sample of a population = its first sample_per_pop neurons (C27); slot = population * sample_per_pop + k
    std::vector<int32_t> sample(N, -1);
    for (size_t p = 0; p < s->pops.size(); ++p)
        for (int k = 0; k < std::min(sample_per_pop, s->pops[p].n); ++k) sample[(size_t)s->pops[p].first + k] = (int32_t)(p * sample_per_pop + k);
    const size_t slots = std::max<size_t>(1, s->pops.size() * (size_t)sample_per_pop);
    uint16_t* bins = nullptr;
    if (!(dev_alloc_t(s, &s->a.st_last, N) && dev_alloc_t(s, &s->a.st_cnt, N) && dev_alloc_t(s, &s->a.st_sum, N) &&
          dev_alloc_t(s, &s->a.st_sumsq, N) && dev_alloc_t(s, &s->d_st_sample, N) && dev_alloc_t(s, &bins, slots * (size_t)max_bins))) {
        s->a.st_cnt = nullptr;
        return fail(s, NG_ERR_OOM, "device allocation failed (statistics)");
    }
    cudaStream_t st = s->stream;
    NG_CUDA(s, cudaMemsetAsync(s->a.st_last, 0xFF, N * 4, st));           // -1: no spike yet
    NG_CUDA(s, cudaMemsetAsync(s->a.st_cnt, 0, N * 4, st));
    NG_CUDA(s, cudaMemsetAsync(s->a.st_sum, 0, N * 8, st));
    NG_CUDA(s, cudaMemsetAsync(s->a.st_sumsq, 0, N * 8, st));
    NG_CUDA(s, cudaMemsetAsync(bins, 0, slots * (size_t)max_bins * 2, st));
    NG_CUDA(s, cudaMemcpyAsync(s->d_st_sample, sample.data(), N * 4, cudaMemcpyHostToDevice, st));
    NG_CUDA(s, cudaStreamSynchronize(st));
    s->a.st_sample = s->d_st_sample; s->a.st_bins = bins;
    s->a.st_start = start_step; s->a.st_bin_steps = bin_steps; s->a.st_max_bins = max_bins;
    s->st_sample_per_pop = sample_per_pop; s->st_slots = (int)slots;
    destroy_graph(s);                                                   // the kernels' argument block changed
    return NG_OK;
}

int32_t ng_get_rate_cv(ng_sim* s, float* rate_hz, float* cv_isi, int64_t count) {
    if (!s || !rate_hz || !cv_isi) return NG_ERR_INVALID_ARG;
    if (!s->prepared || !s->a.st_cnt) return fail(s, NG_ERR_STATE, "statistics are not enabled");
    if (count != s->N) return fail(s, NG_ERR_INVALID_ARG, "count must be the number of neurons");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    Ctl h{};
    int32_t rc = read_ctl(s, &h);
    if (rc) return rc;
    const double T_s = (double)(h.step_u - s->a.st_start) * s->cfg.dt_ms * 1e-3;
    if (!(T_s > 0.0)) return fail(s, NG_ERR_STATE, "no step after the statistics start step yet");
    float *d_rate = nullptr, *d_cv = nullptr;
    if (!(dev_alloc_t(s, &d_rate, (size_t)s->N) && dev_alloc_t(s, &d_cv, (size_t)s->N))) return fail(s, NG_ERR_OOM, "scratch");
    stat_rate_cv_kernel<<<(s->N + 255) / 256, 256, 0, s->stream>>>(s->N, s->a.st_cnt, s->a.st_sum, s->a.st_sumsq, T_s, d_rate, d_cv);
    NG_CUDA(s, cudaMemcpyAsync(rate_hz, d_rate, (size_t)s->N * 4, cudaMemcpyDefault, s->stream));
    NG_CUDA(s, cudaMemcpyAsync(cv_isi, d_cv, (size_t)s->N * 4, cudaMemcpyDefault, s->stream));
    NG_CUDA(s, cudaStreamSynchronize(s->stream));
    dev_free(s, d_rate); dev_free(s, d_cv);
    return NG_OK;
}

int32_t ng_get_correlations(ng_sim* s, int32_t population, float* corr, int64_t capacity, int32_t* n_sample_out, int32_t* n_bins_out) {
    if (!s || !n_sample_out || !n_bins_out || capacity < 0) return NG_ERR_INVALID_ARG;
    *n_sample_out = 0; *n_bins_out = 0;
    if (!s->prepared || !s->a.st_cnt) return fail(s, NG_ERR_STATE, "statistics are not enabled");
    if (population < 0 || population >= (int32_t)s->pops.size()) return fail(s, NG_ERR_INVALID_ARG, "population index");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    Ctl h{};
    int32_t rc = read_ctl(s, &h);
    if (rc) return rc;
    const int ns = std::min(s->st_sample_per_pop, s->pops[population].n);
    const long long full = (h.step_u - s->a.st_start) / s->a.st_bin_steps;            // complete bins only
    const int nb = (int)std::max<long long>(0, std::min<long long>(full, s->a.st_max_bins));
    *n_sample_out = ns; *n_bins_out = nb;
    if (!corr || capacity < (int64_t)ns * ns || ns == 0 || nb == 0) return NG_OK;
    float* d_c = nullptr;
    if (!dev_alloc_t(s, &d_c, (size_t)ns * ns)) return fail(s, NG_ERR_OOM, "scratch");
    stat_corr_kernel<<<s->sm_count * 4, 256, 0, s->stream>>>(s->a.st_bins + (size_t)population * s->st_sample_per_pop * s->a.st_max_bins,
                                                             ns, nb, s->a.st_max_bins, d_c);
    NG_CUDA(s, cudaMemcpyAsync(corr, d_c, (size_t)ns * ns * 4, cudaMemcpyDefault, s->stream));
    NG_CUDA(s, cudaStreamSynchronize(s->stream));
    dev_free(s, d_c);
    return NG_OK;
}

int32_t ng_get_trace(ng_sim* s, uint64_t* out_host, int64_t capacity, int64_t* count_out, int32_t* blocks_out) {
    if (!s || !count_out || !blocks_out || capacity < 0) return NG_ERR_INVALID_ARG;
    *count_out = 0; *blocks_out = 0;
    unsigned long long* t = s->a.trace ? s->a.trace : s->trace_saved;
    if (!t || s->last_persistent_blocks <= 0) return fail(s, NG_ERR_STATE, "no trace: set NG_OPT_TRACE and run step mode 2");
    NG_CUDA(s, cudaSetDevice(s->cfg.device));
    NG_CUDA(s, cudaStreamSynchronize(s->stream));
    const int64_t words = (int64_t)kTraceSteps * s->last_persistent_blocks * kTraceStamps;
    *count_out = words; *blocks_out = s->last_persistent_blocks;
    if (out_host && capacity >= words) NG_CUDA(s, cudaMemcpy(out_host, t, (size_t)words * 8, cudaMemcpyDeviceToHost));
    return NG_OK;
}

}  // extern "C"

// ng_probe: see include/ng.h.  Allocates with cudaMalloc, runs on the legacy stream, frees everything.
extern "C" int32_t ng_probe(int32_t device, int32_t kind, int64_t footprint_bytes, double* per_second_out) {
    if (!per_second_out || kind < 0 || kind > 2 || footprint_bytes < 4096) return NG_ERR_INVALID_ARG;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return NG_ERR_CUDA; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return NG_ERR_CUDA;
    const int blocks = prop.multiProcessorCount * 8, thr = 256;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float ms = 0; double units = 0; int32_t rc = NG_OK;
    float* ring = nullptr; int32_t* tgt = nullptr; float* w = nullptr; int* sink = nullptr;
    const long long n_rec = 1LL << 28;                                  // 2 GiB of records for kinds 0 and 2
    const uint32_t M = (uint32_t)std::min<int64_t>(footprint_bytes / 4, 0x7fffffff);
    do {
        if (cudaMalloc(&sink, 4) != cudaSuccess) { rc = NG_ERR_OOM; break; }
        if (kind == 0) {
            if (cudaMalloc(&tgt, n_rec * 8) != cudaSuccess) { rc = NG_ERR_OOM; break; }
            cudaMemset(tgt, 0, n_rec * 8);
            probe_stream_kernel<<<blocks * 2, thr>>>((const int4*)tgt, n_rec / 2, sink);
            cudaEventRecord(e0);
            probe_stream_kernel<<<blocks * 2, thr>>>((const int4*)tgt, n_rec / 2, sink);
            cudaEventRecord(e1);
            units = (double)n_rec * 8;                                  // bytes
        } else if (kind == 1) {
            if (cudaMalloc(&ring, (size_t)M * 4) != cudaSuccess) { rc = NG_ERR_OOM; break; }
            cudaMemset(ring, 0, (size_t)M * 4);
            probe_red_kernel<<<blocks, thr>>>(ring, M, 100);
            cudaEventRecord(e0);
            probe_red_kernel<<<blocks, thr>>>(ring, M, 2000);
            cudaEventRecord(e1);
            units = (double)blocks * thr * 2000;                        // reductions
        } else {
            if (cudaMalloc(&ring, (size_t)M * 4) != cudaSuccess || cudaMalloc(&tgt, n_rec * 4) != cudaSuccess ||
                cudaMalloc(&w, n_rec * 4) != cudaSuccess) { rc = NG_ERR_OOM; break; }
            cudaMemset(ring, 0, (size_t)M * 4); cudaMemset(w, 0, n_rec * 4);
            probe_fill_targets_kernel<<<blocks, thr>>>(tgt, n_rec, M);
            probe_deliver_kernel<<<blocks, thr>>>((const int4*)tgt, (const float4*)w, ring, n_rec / 32);
            cudaEventRecord(e0);
            probe_deliver_kernel<<<blocks, thr>>>((const int4*)tgt, (const float4*)w, ring, n_rec / 4);
            cudaEventRecord(e1);
            units = (double)n_rec;                                      // events
        }
        if (cudaDeviceSynchronize() != cudaSuccess) { rc = NG_ERR_CUDA; break; }
        cudaEventElapsedTime(&ms, e0, e1);
        *per_second_out = units / (ms * 1e-3);
    } while (0);
    cudaGetLastError();
    cudaFree(ring); cudaFree(tgt); cudaFree(w); cudaFree(sink);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return rc;
}
