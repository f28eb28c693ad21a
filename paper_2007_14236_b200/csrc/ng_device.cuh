// =====================================================================================
// ng_device.cuh — device code of libng.so (sm_100a): Philox, samplers, connection builder,
// fused LIF + Poisson neuron update with spike collection, spike delivery.
// Shares nothing with oracle/ (test infrastructure).  Citations are PAPER.md lines and the
// readings C1..C20 of DESIGN.md.
// =====================================================================================
#pragma once
#include <cooperative_groups.h>
#include <cstdint>
#include <cuda_runtime.h>

#ifndef NG_GC
#define NG_GC __grid_constant__     // kernel parameter block addressable without a local copy (noinline callees take it by reference)
#endif
namespace ng {
namespace cg = cooperative_groups;

// counter word 3 of the Philox stream (C1)
enum : uint32_t { kTagConn = 1, kTagPoisson = 2, kTagInject = 3 };
enum : int32_t { kRuleIndegree = 0, kRuleOutdegree = 1 };
enum : int32_t { kDistConst = 0, kDistNormalClipped = 1, kDistUniformInt = 2 };

constexpr int kMaxPoissonTable = 64;
constexpr int kMaxWindowSteps = 256;     // >= ring_slots (1..255)
constexpr int kTraceSteps = 64;      // the persistent kernels keep the phase stamps of the last kTraceSteps steps
constexpr int kTraceStamps = 16;
constexpr int kUpdateThreads = 256;
constexpr int kDeliverThreads = 256;
constexpr int kChunkRecords = 128;   // records one warp consumes per iteration of the row walk: 32 lanes x 4

struct DistDev { int32_t kind; int32_t pad; double a, b, lo, hi; };

struct CallDev {               // one ng_connect_* call
    int32_t rule, src_first, src_n, tgt_first, tgt_n, K;
    int32_t call_index, port;              // port: receptor port of the targets (0, or 1 = inhibitory conductance of AdEx)
    DistDev w, d;
};

struct AdexDev {               // AdEx constants (fp32 copies of the fp64 host values), Table II symbols
    float g_L, E_L, V_T, inv_DeltaT, gL_DeltaT, inv_C, inv_tau_w, a, b, V_reset, V_peak, E_ex, E_in, inv_tau_syn, I_e;
    float jump;                            // e / tau_syn: conductance-derivative jump per unit weight (reading C22)
    float inv_tol[6];                      // 1 / absolute tolerance of (V, w, g_ex, y_ex, g_in, y_in)
    float h_min;
};
struct PopDev {                // per-population constants of the update (fp32 copies of fp64 host values)
    float P11, P22, P21, P20Ie;            // exact-integration propagators; P20Ie = P20 * I_e
    float E_L, V_th, V_reset, w_ext;
    int32_t refr_steps, n_T;
    uint32_t T[kMaxPoissonTable];          // integer Poisson CDF table (C7)
    int32_t model, pad;                    // 0 = LIF (iaf_psc_exp), 1 = AdEx with alpha conductances
    AdexDev ax;
};

// Device-resident control block; see ng.cu for the update/deliver handshake.  Words with different traffic live on
// different 128-byte lines: the barrier counter is polled by every CTA while late CTAs still append spikes
// (atomics on spike_cnt) and count events — on one line those requests queue at the same L2 slice.
struct alignas(128) BarWord { unsigned long long v; };   // one barrier word per 128-byte line: polls and arrivals of different
                                                           // barriers do not queue at one L2 slice
struct Ctl {
    // line 0: step bookkeeping, written once per step by one thread
    alignas(128) long long step_u;         // written by deliver, read by update: index of the next step
    long long step_d;                      // written by update, read by deliver: index of the step being delivered
    unsigned long long rec_total[2];       // spikes recorded before step of this parity
    unsigned long long spikes;
    int32_t err_delay;                     // builder: a drawn delay fell outside [1, D]
    int32_t max_row_records;               // builder: longest padded row
    unsigned long long n_padded;           // builder: total records stored
    int32_t pending;                       // pipelined step kernel: the rest pass of step step_u - 1 is outstanding
    int32_t slot;                          // step_u mod Dr, kept next to step_u so no kernel divides 64-bit integers
    int32_t slot_d;                        // step_d mod Dr: written by update, read by deliver (like step_d) — the delivery
                                           // kernel's bookkeeping advances `slot` while later CTAs of the same launch still start
    int32_t err_window;                    // spike-buffer backend: the spike window overflowed its capacity
    uint32_t n_long_groups;                // builder: (source, delay) groups longer than kSortMax, listed for the CTA-wide sort
    int32_t err_queue;                     // event-queue backend: a queue overflowed its capacity (events were dropped)
    unsigned long long win_tail;           // pipelined spike-buffer backend (kernel 6): next free position of the spike window
    int32_t err_xchg;                      // target-sharded mode: a peer's spike list did not arrive (bounded wait expired)
    unsigned long long n_records;          // builder: records stored on this shard (unpadded)
    // line 1: spike counters (atomics of the appending warps / CTAs)
    alignas(128) int32_t spike_cnt[4];     // length of the spike array of step n, indexed n & 3 (the list itself by n & 1)
    int32_t spike_cnt8[8];                 // split kernel: the same, indexed n & 7 (its warp groups run up to two steps apart)
    // line 2: event counter (one atomic per CTA and step)
    alignas(128) unsigned long long events;
    // line 3: grid barrier of the persistent kernels, and the ticket of the stand-alone pipelined kernel
    alignas(128) unsigned long long bar;   // arrivals at the grid barrier
    unsigned int ticket;                   // CTAs that finished the current step
    BarWord bar_plane[2];                  // split kernel: CTAs whose reductions of a phase are all issued and acknowledged, and
    BarWord bar_list[2];                   // split kernel: CTAs that have appended their spikes of a step to the global spike array,
                                           // one word per step parity each (a CTA may arrive for step n + 1 while another still
                                           // waits for step n to be complete: on one word its arrival would stand in for a missing one;
                                           // it cannot arrive for step n + 2 before step n is complete)
    // line 4 ..: spike-buffer backend
    alignas(128) unsigned long long win_start[kMaxWindowSteps + 1];   // absolute position in the spike window of the first
                                           // spike of step s, at index s mod (D+1); [s+1] = its end
};

// ---------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11).  key = 64-bit seed (lo, hi), C1.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2,
                                               uint32_t c3) {
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += W0; k1 += W1;
    }
    return make_uint4(c0, c1, c2, c3);
}

__device__ __forceinline__ int32_t mulhi_range(uint32_t x, uint32_t n) {   // DESIGN.md C2
    return (int32_t)__umulhi(x, n);
}

// One connection draw, a pure function of (seed, call, endpoint, k) — DESIGN.md C1-C5.
// Every fp64 operation is an explicitly rounded intrinsic so no FMA contraction can change a bit.
struct Draw { int32_t src, tgt, delay; float w; };

template <bool kNeedWeight>
__device__ __forceinline__ Draw draw_connection(const CallDev& c, uint32_t seed_lo, uint32_t seed_hi, int32_t endpoint,
                                                int32_t k) {
    const uint4 x = philox4x32_10(seed_lo, seed_hi, (uint32_t)k, (uint32_t)endpoint, (uint32_t)c.call_index, kTagConn);
    Draw out;
    if (c.rule == kRuleIndegree) {
        out.tgt = endpoint;
        out.src = c.src_first + mulhi_range(x.x, (uint32_t)c.src_n);
    } else {
        out.src = endpoint;
        out.tgt = c.tgt_first + mulhi_range(x.x, (uint32_t)c.tgt_n);
    }
    double z_w = 0.0, z_d = 0.0;
    const bool normal_w = kNeedWeight && c.w.kind == kDistNormalClipped;
    const bool normal_d = c.d.kind == kDistNormalClipped;
    if (normal_w || normal_d) {                                          // C4: fp64 Box-Muller from (x1, x2)
        const double u1 = __dmul_rn(__dadd_rn((double)x.y, 0.5), 1.0 / 4294967296.0);
        const double u2 = __dmul_rn(__dadd_rn((double)x.z, 0.5), 1.0 / 4294967296.0);
        const double r = sqrt(__dmul_rn(-2.0, log(u1)));
        const double a = __dmul_rn(6.283185307179586476925286766559, u2);
        double sa, ca;
        sincos(a, &sa, &ca);
        z_w = __dmul_rn(r, ca);
        z_d = __dmul_rn(r, sa);
    }
    out.w = 0.f;
    if (kNeedWeight) {
        double w;
        if (c.w.kind == kDistConst) w = c.w.a;
        else if (c.w.kind == kDistNormalClipped) {
            w = __dadd_rn(c.w.a, __dmul_rn(c.w.b, z_w));
            if (w < c.w.lo) w = c.w.lo;
            if (w > c.w.hi) w = c.w.hi;
        } else {
            const double span = __dadd_rn(__dsub_rn(c.w.hi, c.w.lo), 1.0);
            w = __dadd_rn(c.w.lo, (double)(((uint64_t)x.w * (uint64_t)span) >> 32));
        }
        out.w = (float)w;                                                // the record stores fp32
    }
    long long d;
    if (c.d.kind == kDistConst) d = (long long)c.d.a;
    else if (c.d.kind == kDistUniformInt) {                              // C5
        const uint64_t span = (uint64_t)((long long)c.d.hi - (long long)c.d.lo + 1);
        d = (long long)c.d.lo + (long long)(((uint64_t)x.w * span) >> 32);
    } else {                                                             // C5: round half up, then clip
        double f = floor(__dadd_rn(__dadd_rn(c.d.a, __dmul_rn(c.d.b, z_d)), 0.5));
        if (f < c.d.lo) f = c.d.lo;
        if (f > c.d.hi) f = c.d.hi;
        d = (long long)f;
    }
    out.delay = (int32_t)d;
    return out;
}

// ---------------------------------------------------------------------------------------
// a0. Connection builder (PAPER.md:37 rules, built in GPU memory as PAPER.md:292 proposes).
//   pass 1  count records per (source, delay)                    build_count_kernel
//           row lengths (padded to 4), exclusive scan            build_rowlen_kernel, scan kernels
//           group offsets inside each row                        build_groups_kernel
//   pass 2  regenerate every draw and scatter it into its group  build_fill_kernel
// The rows come out source-major with groups of equal delay in increasing delay order — the
// layout of PAPER.md:69 / Fig. 1(a).
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
build_count_kernel(const CallDev* __restrict__ calls, int call_idx, uint32_t seed_lo, uint32_t seed_hi, int D,
                   uint32_t* __restrict__ cnt, Ctl* __restrict__ ctl, int32_t id_first, int32_t id_n) {
    const CallDev c = calls[call_idx];
    // target-sharded build: this GPU stores the connections whose TARGET is in [id_first, id_first + id_n).
    // A draw is a pure function of (seed, call, endpoint, k), so the shard's structure is the one-GPU structure
    // restricted to those targets.  Fixed in-degree: the endpoint is the target, so only local endpoints are drawn.
    const int32_t e_first = c.rule == kRuleIndegree ? max(c.tgt_first, id_first) : c.src_first;
    const int32_t e_n = c.rule == kRuleIndegree ? max(0, min(c.tgt_first + c.tgt_n, id_first + id_n) - e_first) : c.src_n;
    const long long total = (long long)e_n * c.K;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += stride) {
        const int32_t e = e_first + (int32_t)(idx / c.K);
        const int32_t k = (int32_t)(idx % c.K);
        const Draw dr = draw_connection<false>(c, seed_lo, seed_hi, e, k);
        if (dr.tgt < id_first || dr.tgt >= id_first + id_n) continue;
        if (dr.delay < 1 || dr.delay > D) { ctl->err_delay = 1; continue; }
        atomicAdd(&cnt[(size_t)dr.src * D + (dr.delay - 1)], 1u);
    }
}

// row_len[j] = out-degree of j padded to a multiple of 4 records (so every row starts 16-byte aligned
// in the tgt / w arrays and can be read with 128-bit loads)
__global__ void build_rowlen_kernel(const uint32_t* __restrict__ cnt, int N, int D, long long* __restrict__ row_len,
                                    Ctl* __restrict__ ctl) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    int len = 0;
    int deg = 0;
    if (j < N) {
        for (int d = 0; d < D; ++d) deg += (int)cnt[(size_t)j * D + d];
        len = (deg + 3) & ~3;
        row_len[j] = len;
    }
    // block max and block sum -> one atomic each per block
    __shared__ int smax;
    __shared__ unsigned long long ssum;
    if (threadIdx.x == 0) { smax = 0; ssum = 0; }
    __syncthreads();
    atomicMax(&smax, len);
    if (deg) atomicAdd(&ssum, (unsigned long long)deg);
    __syncthreads();
    if (threadIdx.x == 0) { atomicMax(&ctl->max_row_records, smax); if (ssum) atomicAdd(&ctl->n_records, ssum); }
}

// Exclusive scan of int64 values, one CTA of 1024 threads walking the array tile by tile.  N <= a few 1e6
// and this runs once, so a single-CTA scan is simple and fast enough (~1 ms at N = 1e6).
__global__ void __launch_bounds__(1024)
scan_exclusive_kernel(const long long* __restrict__ in, long long* __restrict__ out, int N, Ctl* __restrict__ ctl) {
    __shared__ long long warp_sum[32];
    __shared__ long long carry_s;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < N; base += 1024) {
        const int i = base + threadIdx.x;
        const long long v = i < N ? in[i] : 0;
        long long x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const long long y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_sum[wid] = x;
        __syncthreads();
        if (wid == 0) {
            long long s = warp_sum[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const long long y = __shfl_up_sync(0xffffffffu, s, o);
                if (lane >= o) s += y;
            }
            warp_sum[lane] = s;
        }
        __syncthreads();
        const long long carry = carry_s;
        const long long incl = x + (wid > 0 ? warp_sum[wid - 1] : 0) + carry;
        if (i < N) out[i] = incl - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[N] = carry_s; ctl->n_padded = (unsigned long long)carry_s; }
}

// grp_rel[j*(D+1) + d] = offset inside row j of the first record with delay d+1; entry D = out-degree.
// Also clears cnt so that pass 2 can use it as the per-group fill cursor.
__global__ void build_groups_kernel(uint32_t* __restrict__ cnt, int N, int D, uint32_t* __restrict__ grp_rel) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    uint32_t run = 0;
    for (int d = 0; d < D; ++d) {
        grp_rel[(size_t)j * (D + 1) + d] = run;
        run += cnt[(size_t)j * D + d];
        cnt[(size_t)j * D + d] = 0;
    }
    grp_rel[(size_t)j * (D + 1) + D] = run;
}

// row_info[j] = (first record, out-degree, padded length) of row j in one 16-byte word: the thread that detects a
// spike fetches everything delivery needs with a single load.
// deg = out-degree (the stored row is padded to a multiple of 4 records), d1 = records with delay 1 (the first d1 of the row)
struct __align__(16) RowInfo { long long r0; int32_t deg; int32_t d1; };
__host__ __device__ __forceinline__ int32_t padded_len(int32_t deg) { return (deg + 3) & ~3; }
__global__ void build_row_info_kernel(int N, int D, const long long* __restrict__ row_off, const uint32_t* __restrict__ grp_rel,
                                      RowInfo* __restrict__ row_info) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    RowInfo r;
    r.r0 = row_off[j]; r.deg = (int32_t)grp_rel[(size_t)j * (D + 1) + D]; r.d1 = (int32_t)grp_rel[(size_t)j * (D + 1) + 1];
    row_info[j] = r;
}

__global__ void __launch_bounds__(256)
build_fill_kernel(const CallDev* __restrict__ calls, int call_idx, uint32_t seed_lo, uint32_t seed_hi, int D,
                  uint32_t* __restrict__ cursor, const long long* __restrict__ row_off,
                  const uint32_t* __restrict__ grp_rel, int32_t* __restrict__ tgt, float* __restrict__ w,
                  uint8_t* __restrict__ dly, int n_neurons, int32_t id_first) {
    const CallDev c = calls[call_idx];
    const int32_t id_n = n_neurons;                           // n_neurons = neurons of this shard
    const int32_t e_first = c.rule == kRuleIndegree ? max(c.tgt_first, id_first) : c.src_first;
    const int32_t e_n = c.rule == kRuleIndegree ? max(0, min(c.tgt_first + c.tgt_n, id_first + id_n) - e_first) : c.src_n;
    const long long total = (long long)e_n * c.K;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += stride) {
        const int32_t e = e_first + (int32_t)(idx / c.K);
        const int32_t k = (int32_t)(idx % c.K);
        const Draw dr = draw_connection<true>(c, seed_lo, seed_hi, e, k);
        if (dr.tgt < id_first || dr.tgt >= id_first + id_n) continue;
        if (dr.delay < 1 || dr.delay > D) continue;
        const uint32_t p = atomicAdd(&cursor[(size_t)dr.src * D + (dr.delay - 1)], 1u);
        const long long pos = row_off[dr.src] + grp_rel[(size_t)dr.src * (D + 1) + (dr.delay - 1)] + p;
        tgt[pos] = dr.tgt - id_first + c.port * n_neurons;  // local target index; receptor port folded into the ring column
        w[pos] = dr.w;
        dly[pos] = (uint8_t)dr.delay;
    }
}

// Order the records of every (source, delay) group by (target, weight bits): the fill order above depends on
// atomic arrival order; after this pass the structure is a deterministic function of the seed.
// One warp per group; groups are short (1..~1e3 records), so an in-place odd-even transposition over
// lane-strided elements is enough.  Groups longer than kSortMax records (out-degree >= 1000 with a constant delay,
// say) are listed in `long_list` and sorted by build_sort_long_groups_kernel, one CTA each.
constexpr int kSortMax = 768;    // 8 warps x 768 x 8 B = 48 KB of static shared memory
__global__ void __launch_bounds__(256)
build_sort_groups_kernel(int N, int D, const long long* __restrict__ row_off, const uint32_t* __restrict__ grp_rel,
                         int32_t* __restrict__ tgt, float* __restrict__ w, long long* __restrict__ long_list,
                         uint32_t long_cap, Ctl* __restrict__ ctl) {
    __shared__ unsigned long long keys[8][kSortMax];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const long long n_groups = (long long)N * D;
    const long long warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long g = (((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5); g < n_groups; g += warps) {
        const int j = (int)(g / D), d = (int)(g % D);
        const uint32_t a = grp_rel[(size_t)j * (D + 1) + d], b = grp_rel[(size_t)j * (D + 1) + d + 1];
        const int len = (int)(b - a);
        if (len < 2) continue;
        if (len > kSortMax) {
            if (lane == 0) { const uint32_t k = atomicAdd(&ctl->n_long_groups, 1u); if (k < long_cap) long_list[k] = g; }
            continue;
        }
        const long long base = row_off[j] + a;
        unsigned long long* K = keys[wib];
        for (int i = lane; i < len; i += 32)
            K[i] = ((unsigned long long)(uint32_t)tgt[base + i] << 32) | (unsigned long long)__float_as_uint(w[base + i]);
        __syncwarp();
        for (int pass = 0; pass < len; ++pass) {
            for (int i = (pass & 1) + 2 * lane; i + 1 < len; i += 64) {
                const unsigned long long x = K[i], y = K[i + 1];
                if (x > y) { K[i] = y; K[i + 1] = x; }
            }
            __syncwarp();
        }
        for (int i = lane; i < len; i += 32) {
            tgt[base + i] = (int32_t)(uint32_t)(K[i] >> 32);
            w[base + i] = __uint_as_float((uint32_t)K[i]);
        }
        __syncwarp();
    }
}

// Long groups: one CTA per listed group sorts it in place in global memory with a bitonic network whose merges all run
// in ascending direction (first stage of a merge of size k pairs i with i ^ (k - 1), the others i with i ^ j), so a
// length that is not a power of two needs no padding: the cells beyond the end behave as +infinity and never move.
__global__ void __launch_bounds__(1024)
build_sort_long_groups_kernel(int D, const long long* __restrict__ row_off, const uint32_t* __restrict__ grp_rel,
                              int32_t* __restrict__ tgt, float* __restrict__ w, const long long* __restrict__ long_list,
                              uint32_t long_cap, const Ctl* __restrict__ ctl) {
    const uint32_t n_long = min(ctl->n_long_groups, long_cap);
    for (uint32_t k = blockIdx.x; k < n_long; k += gridDim.x) {
        const long long g = long_list[k];
        const int j = (int)(g / D), d = (int)(g % D);
        const uint32_t a = grp_rel[(size_t)j * (D + 1) + d], b = grp_rel[(size_t)j * (D + 1) + d + 1];
        const uint32_t len = b - a;
        int32_t* __restrict__ T = tgt + row_off[j] + a;
        float* __restrict__ W = w + row_off[j] + a;
        auto cmpx = [&](uint32_t i, uint32_t l) {              // ascending compare-exchange of cells i < l < len
            const unsigned long long x = ((unsigned long long)(uint32_t)T[i] << 32) | __float_as_uint(W[i]);
            const unsigned long long y = ((unsigned long long)(uint32_t)T[l] << 32) | __float_as_uint(W[l]);
            if (x > y) {
                T[i] = (int32_t)(uint32_t)(y >> 32); W[i] = __uint_as_float((uint32_t)y);
                T[l] = (int32_t)(uint32_t)(x >> 32); W[l] = __uint_as_float((uint32_t)x);
            }
        };
        for (uint32_t kk = 2; (kk >> 1) < len; kk <<= 1) {
            for (uint32_t i = threadIdx.x; i < len; i += blockDim.x) {
                const uint32_t l = i ^ (kk - 1);
                if (l > i && l < len) cmpx(i, l);
            }
            __syncthreads();
            for (uint32_t jj = kk >> 2; jj > 0; jj >>= 1) {
                for (uint32_t i = threadIdx.x; i < len; i += blockDim.x) {
                    const uint32_t l = i ^ jj;
                    if (l > i && l < len) cmpx(i, l);
                }
                __syncthreads();
            }
        }
    }
}

// ---------------------------------------------------------------------------------------
// Warp-aggregated append to the spike array (Fig. 1b: "the spike is sent to the spike
// array"; its maximum size is the number of nodes).  One atomicAdd per warp that holds a spike.
// Every lane of the warp must call this.  Next to the id the entry carries the row bounds of the spiking neuron
// (one 16-byte load from row_info), so delivery starts from the entry without a second dependent lookup.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ RowInfo ld_row_info(const RowInfo* p) {
    const int4 v = __ldg(reinterpret_cast<const int4*>(p));
    RowInfo r;
    r.r0 = (long long)(((unsigned long long)(uint32_t)v.y << 32) | (uint32_t)v.x); r.deg = v.z; r.d1 = v.w;
    return r;
}
__device__ __forceinline__ void st_row_info(RowInfo* p, const RowInfo& r) {
    *reinterpret_cast<int4*>(p) = make_int4((int)(uint32_t)(unsigned long long)r.r0, (int)(uint32_t)((unsigned long long)r.r0 >> 32), r.deg, r.d1);
}
// L2 eviction priorities: connection records are read once per spike and never again soon (evict first), the input
// ring is written by the reductions and read back by the update a few steps later (evict last), so that streaming
// gigabytes of records does not push ring planes out of the 126 MB L2.
#if defined(NG_EVICT_HINTS)
__device__ __forceinline__ uint64_t l2_policy_stream() { uint64_t p; asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p)); return p; }
__device__ __forceinline__ uint64_t l2_policy_keep() { uint64_t p; asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p)); return p; }
#endif
__device__ __forceinline__ void red_add_f32(float* addr, float v) {
#if defined(NG_EVICT_HINTS) && NG_EVICT_HINTS >= 2
    asm volatile("red.global.add.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(addr), "f"(v), "l"(l2_policy_keep()) : "memory");
#else
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
#endif
}
// input cell of the ring: read at L2 (it is written by red.global from other SMs) and cleared
__device__ __forceinline__ float ld_plane(const float* p) {
    float v;
#if defined(NG_EVICT_HINTS) && NG_EVICT_HINTS >= 3
    asm volatile("ld.global.cg.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(l2_policy_keep()));
#else
    asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(v) : "l"(p));
#endif
    return v;
}
__device__ __forceinline__ void clear_plane(float* p) {
#if defined(NG_EVICT_HINTS) && NG_EVICT_HINTS >= 3
    asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(0.f), "l"(l2_policy_keep()) : "memory");
#else
    *p = 0.f;
#endif
}
__device__ __forceinline__ int4 ld_stream_s32x4(const int32_t* p) {
    int4 r;
#if defined(NG_EVICT_HINTS)
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.s32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p), "l"(l2_policy_stream()));
#else
    asm("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
#endif
    return r;
}
__device__ __forceinline__ float4 ld_stream_f32x4(const float* p) {
    float4 r;
#if defined(NG_EVICT_HINTS)
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p), "l"(l2_policy_stream()));
#else
    asm("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
#endif
    return r;
}
__device__ __forceinline__ uint32_t ld_stream_u32(const void* p) {
    uint32_t r;
#if defined(NG_EVICT_HINTS)
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.u32 %0, [%1], %2;" : "=r"(r) : "l"(p), "l"(l2_policy_stream()));
#else
    asm("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(r) : "l"(p));
#endif
    return r;
}

// TMA-unit bulk prefetch into L2 (no destination): p 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void prefetch_l2_bulk(const void* p, uint32_t bytes) {
#if defined(NG_EVICT_HINTS)
    uint64_t pol;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("cp.async.bulk.prefetch.L2.global.L2::cache_hint [%0], %1, %2;" ::"l"(p), "r"(bytes), "l"(pol) : "memory");
#else
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
#endif
}
struct StepArgs;
__device__ __forceinline__ void prefetch_row(const StepArgs& a, const RowInfo& r);

struct StepArgs {
    int32_t N, D;                // N = neurons of THIS shard (all neurons on one GPU); D = ring_slots = largest legal delay
    int32_t NS, id_first;        // NS = sources = neurons of the whole network (rows, spike array); global id of local
                                 // neuron i = id_first + i.  One GPU: NS = N, id_first = 0.
    unsigned char* xchg[16];     // target-sharded mode: receive buffers of all ranks as seen from this device ([rank] = own)
    int32_t xchg_rank, xchg_world, xchg_cap, xchg_pad;
    int32_t Dr, n_pops;          // Dr = D + 1 planes are stored (see update_phase); number of populations
    int32_t NR, pad_nr;          // ring row length = N * receptor ports (2 as soon as an AdEx population exists):
                                 // plane of (slot, port) = ring + (slot * NR + port * N); records store target + port * N
    float *ax_w, *ax_gx, *ax_yx, *ax_gi, *ax_yi, *ax_h;     // AdEx state, [N] each (nullptr without AdEx populations)
    uint32_t seed_lo, seed_hi;
    // neuron state (SoA) and parameters
    float* V; float* I; int32_t* refr; const uint8_t* pop_of; const PopDev* pops;
    float* ring;                 // [Dr][N] slot-major
    float* last_input;           // [N] or nullptr (NG_DEBUG_INPUT)
    // spike array, double-buffered by step parity, and the spike record
    int32_t* spike_list;         // [2][N]
    RowInfo* spike_row;          // [2][N] row bounds of spike_list's entries (same index)
    const RowInfo* row_info;     // [N]
    int32_t prefetch;            // 1: a spiking thread bulk-prefetches its row into L2 (row-walk kernels)
    uint8_t* pois_k;             // [N] Poisson counts of the next step (persistent pipelined kernel)
    // on-device spike statistics, nullptr until ng_enable_statistics: accumulated by the thread that
    // detects the spike — a neuron spikes at most once per step and always in one thread, so no atomics are needed
    int32_t* st_last; int32_t* st_cnt; double* st_sum; double* st_sumsq;       // [N]: last spike step, spikes, sum ISI, sum ISI^2
    const int32_t* st_sample; uint16_t* st_bins;                                // [N] sample slot or -1; [slots][st_max_bins] binned trains
    long long st_start; int32_t st_bin_steps, st_max_bins;
    int32_t* win_id;             // spike-buffer backend (delivery kernel 4): circular log of the spikes of the last D steps
    long long win_cap;           //   its capacity in entries; nullptr / 0 for the ring backends
    int2* q_ev;                  // event-queue backend (delivery kernel 5): [D][q_cap] (target, weight bits) by arrival step mod D
    unsigned long long* q_tail;  //   events appended to the queue of each arrival slot, one counter per 128-byte line
    long long q_cap;             //   capacity of one queue in events (even); nullptr / 0 for the other backends
    unsigned long long* trace;   // NG_OPT_TRACE: [kTraceSteps][gridDim.x][kTraceStamps] %globaltimer stamps, or nullptr
    int32_t* rec_step; int32_t* rec_id; long long rec_cap;   // rec_cap = 0: recording off
    // connection structure
    const long long* row_off; const uint32_t* grp_rel;
    const int32_t* tgt; const float* w; const uint8_t* dly;
    Ctl* ctl;
    int32_t bypass; uint32_t inject_thr;
    float dt_ms; int32_t has_adex;
    int32_t max_row_chunks;      // ceil(longest padded row / kChunkRecords)
    int32_t mean_row_records;    // mean padded row length (>= 1): picks the item size of delivery kernel 1
};

// Spike statistics at spike time: per neuron the spike count and the first two moments of the
// inter-spike interval (in steps, exact in fp64), and for the sampled neurons the spike train re-binned to st_bin_steps.
__device__ __forceinline__ void stat_on_spike(const StepArgs& a, int i, long long n) {
    if (!a.st_cnt || n < a.st_start) return;
    const int last = a.st_last[i];
    a.st_last[i] = (int)n;
    a.st_cnt[i] += 1;
    if (last >= 0) { const double isi = (double)((int)n - last); a.st_sum[i] += isi; a.st_sumsq[i] += isi * isi; }
    const int slot = a.st_sample[i];
    if (slot >= 0) {
        const long long bin = (n - a.st_start) / a.st_bin_steps;
        if (bin < a.st_max_bins) a.st_bins[(size_t)slot * a.st_max_bins + bin] += 1;
    }
}

// The records of a spiking row are requested from DRAM the moment the spike is detected: by the time the delivery
// phase (after the grid barrier / kernel boundary) asks for them they are L2 hits.  Pieces of at most 32 KB.
__device__ __forceinline__ void prefetch_row(const StepArgs& a, const RowInfo& r) {
    const int len = padded_len(r.deg);
    const long long bytes4 = (long long)len * 4;
    const uint32_t head = (uint32_t)(((long long)r.d1 * 4 + 15) & ~15LL);      // delay-1 records: needed first (pipelined kernel 3)
    if (head > 0 && head < 32768) {
        prefetch_l2_bulk(reinterpret_cast<const char*>(a.tgt + r.r0), head);
        prefetch_l2_bulk(reinterpret_cast<const char*>(a.w + r.r0), head);
    }
    for (long long o = 0; o < bytes4; o += 32768) {
        const uint32_t b = (uint32_t)(bytes4 - o < 32768 ? bytes4 - o : 32768);
        prefetch_l2_bulk(reinterpret_cast<const char*>(a.tgt + r.r0) + o, b);
        prefetch_l2_bulk(reinterpret_cast<const char*>(a.w + r.r0) + o, b);
    }
    const long long d0 = r.r0 & ~15LL, d1 = (r.r0 + len + 15) & ~15LL;       // delay bytes, 16-byte grid
    for (long long o = d0; o < d1; o += 32768)
        prefetch_l2_bulk(a.dly + o, (uint32_t)(d1 - o < 32768 ? d1 - o : 32768));
}

// `rec_base` = number of spikes recorded before step n: the spiking thread also writes the spike record (a2,
// PAPER.md:181 "all spike times of all neurons recorded").  The atomic is issued before the row lookup and the
// prefetches so that all three overlap.
__device__ __forceinline__ void append_spike(const StepArgs& a, bool spk, int32_t i_local, long long n, unsigned long long rec_base,
                                             unsigned long long win_base = 0) {
    const unsigned m = __ballot_sync(0xffffffffu, spk);
    if (m == 0) return;
    const int32_t id = a.id_first + i_local;                  // the spike array, the record and the rows use global ids
    const int lane = threadIdx.x & 31;
    const int leader = __ffs(m) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(&a.ctl->spike_cnt[n & 3], __popc(m));
    RowInfo r;
    if (spk) { r = ld_row_info(a.row_info + id); if (a.prefetch && !a.win_id) prefetch_row(a, r); }
    base = __shfl_sync(0xffffffffu, base, leader);
    if (spk) {
        const int idx = base + __popc(m & ((1u << lane) - 1u));
        const size_t k = (size_t)(n & 1) * a.NS + idx;
        a.spike_list[k] = id;
        st_row_info(a.spike_row + k, r);
        const unsigned long long pos = rec_base + (unsigned long long)idx;
        if (pos < (unsigned long long)a.rec_cap) { a.rec_id[pos] = id; a.rec_step[pos] = (int32_t)n; }
        if (a.win_id) a.win_id[(win_base + (unsigned long long)idx) % (unsigned long long)a.win_cap] = id;
        stat_on_spike(a, i_local, n);
    }
}

// ---------------------------------------------------------------------------------------
// a1 + a2. Neuron update fused with the Poisson drive and spike collection — one thread per neuron.
//   PAPER.md:93-102 Eqs. (1)-(2), exact integration PAPER.md:37; order of operations DESIGN.md C11:
//     in  = ring[n mod D][i], slot cleared                                       (C9)
//     k   ~ Poisson(lambda_pop) from Philox(seed; i, n, POISSON)                 (C7)
//     V  <- E_L + P22 (V - E_L) + P21 I + P20 I_e    if not refractory, else refr--
//     I  <- P11 I + in + w_ext k
//     V >= V_th: spike, V <- V_reset, refr <- t_ref/h
// `gtid`/`gthreads` let the same body serve the stand-alone kernel and the persistent kernel.
// ---------------------------------------------------------------------------------------
// One neuron, one step.  `P` is the population table (global memory, or the CTA's shared-memory copy).
// The ring stores Dr = D + 1 planes: the plane consumed here (n mod Dr) can then never be a delivery target of
// step n (targets are (n + d) mod Dr, 1 <= d <= D), so the fused step kernel may deliver a spike while other
// CTAs are still consuming their inputs.
// Split in two so that the spike is known as early as possible: neuron_early needs only V, I_syn, refr (one memory
// round trip); the caller then starts everything that depends on the spike (row lookup, L2 prefetch of the row,
// counters) and neuron_late — Philox, Poisson count, I_syn update: most of the arithmetic — overlaps those latencies.
// The arithmetic and its order are exactly those of the list above (V uses I before its update).
struct NeuronRegs { float in, I; int pi, kq; float in1; bool adex; bool pending; bool spiked; float t; };     // kq: Poisson count computed ahead of time, or 0xff


// DESIGN.md C7: k = #{m : x0 >= T[m]}, x0 from Philox(seed; i, n, POISSON); T is non-decreasing.  A pure function of
// (seed, i, n): the persistent pipelined kernel evaluates it for step n+1 while it waits at the grid barrier.
__device__ __forceinline__ int poisson_count(const StepArgs& a, const PopDev* __restrict__ p, long long n, int i) {
    int k = 0;
    const int nT = p->n_T;
    if (nT > 0) {
        const uint4 x = philox4x32_10(a.seed_lo, a.seed_hi, (uint32_t)i, (uint32_t)n, (uint32_t)(n >> 32), kTagPoisson);
        while (k < nT && x.x >= p->T[k]) ++k;
    }
    return k;
}

// ---------------------------------------------------------------------------------------
// AdEx neuron with conductance-based alpha synapses — the model of the paper's balanced network:
//   Eq. (3)  C dV/dt = -g_L (V - E_L) + g_L Delta_T exp((V - V_T)/Delta_T) + I_syn - w + I_e
//   Eq. (4)  I_syn = sum_i g_i (E_rev,i - V)                 (sign: DESIGN.md reading C21)
//   Eq. (5)  tau_w dw/dt = a (V - E_L) - w;   spike: V -> V_r, w -> w + b
//   alpha conductances g' = -g/tau + y, y' = -y/tau, a spike of weight W raises y by W e / tau   (C22)
// integrated with "the 5th order Runge-Kutta method with adaptive control of the step size": embedded
// Cash-Karp 5(4), controller and spike rule as readings C23-C25 state them.  fp32 throughout.
// ---------------------------------------------------------------------------------------
struct AdexY { float V, w, gx, yx, gi, yi; };
struct AdexK { float V, w; };

// Right-hand side of Eqs. (3) and (5) for given conductances (Eq. (4) with reading C21).
__device__ __forceinline__ AdexK adex_rhs_vw(const AdexDev& p, float Vs, float ws, float gx, float gi) {
    const float V = fminf(Vs, p.V_peak);                                            // C24
    const float I_spike = p.gL_DeltaT * __expf((V - p.V_T) * p.inv_DeltaT);
    const float I_syn = fmaf(gx, p.E_ex - V, gi * (p.E_in - V));                    // C21
    AdexK f;
    f.V = (fmaf(-p.g_L, V - p.E_L, I_spike) + I_syn - ws + p.I_e) * p.inv_C;
    f.w = (p.a * (V - p.E_L) - ws) * p.inv_tau_w;
    return f;
}

// One time step of one neuron (C23, C24), resumable: at most max_iter attempts of the controller loop; t (time reached
// inside the step) and spiked carry over.  Returns true when the step is complete.  The pipelined kernel gives every
// neuron ONE attempt in its own lane (99 % finish: the sub-step is the whole time step) and collects the others —
// neurons on the exponential upswing, up to thirty sub-steps — in a CTA list that is worked off by dense warps
// afterwards, so that a warp does not wait for its slowest lane.
//
// The embedded Cash-Karp 5(4) step is applied to the six-component system, as the oracle does, but only V and w carry
// their six stage derivatives in registers: the alpha-conductance pair u = (g, y) of a port obeys the LINEAR autonomous
// system u' = A u, A = -1/tau I + N (N nilpotent), for which every Runge-Kutta stage value is a polynomial in x = -h/tau
// applied to u:   y_i = s_i(x) y,   g_i = s_i(x) g + h s_i'(x) y,
// with s_1 = 1, s_i(x) = 1 + x sum_{j<i} b_ij s_j(x); the 5th-order result uses p(x) = 1 + x sum_j c_j s_j(x) and the
// error estimate e(x) = x sum_j (c_j - c*_j) s_j(x) in the same way.  (Coefficients below: exact rationals of the
// Cash-Karp tableau.)  Same arithmetic as the six-component stage loop up to fp32 rounding, 24 fewer live registers — the
// 64-register budget of two 512-thread CTAs per SM is then met without local-memory spills.
template <bool kOneAttempt>
__device__ __forceinline__ bool adex_advance(const AdexDev& p, AdexY& y, float& h_int, float& t, bool& spiked, float h_step) {
    for (int it = 0; t < h_step; ++it) {
        if (kOneAttempt && it >= 1) return false;
        const float h = fmaxf(h_int, p.h_min);
        const bool clipped = h > h_step - t;
        const float ht = clipped ? h_step - t : h;
        const float x = -ht * p.inv_tau_syn;
        // stage conductances g_i = s_i(x) g + h s_i'(x) y of both ports
#define NG_G(si, dsi) const float s_ = (si), hd_ = ht * (dsi); const float gx_ = fmaf(s_, y.gx, hd_ * y.yx), gi_ = fmaf(s_, y.gi, hd_ * y.yi);
        const AdexK k1 = adex_rhs_vw(p, y.V, y.w, y.gx, y.gi);
        AdexK k2, k3, k4, k5, k6;
        { NG_G(fmaf(0.2f, x, 1.f), 0.2f)
          k2 = adex_rhs_vw(p, fmaf(ht, 0.2f * k1.V, y.V), fmaf(ht, 0.2f * k1.w, y.w), gx_, gi_); }
        { NG_G(fmaf(x, fmaf(0.045f, x, 0.3f), 1.f), fmaf(0.09f, x, 0.3f))
          k3 = adex_rhs_vw(p, fmaf(ht, 0.075f * k1.V + 0.225f * k2.V, y.V), fmaf(ht, 0.075f * k1.w + 0.225f * k2.w, y.w), gx_, gi_); }
        { NG_G(fmaf(x, fmaf(x, fmaf(0.054f, x, 0.18f), 0.6f), 1.f), fmaf(x, fmaf(0.162f, x, 0.36f), 0.6f))
          k4 = adex_rhs_vw(p, fmaf(ht, 0.3f * k1.V - 0.9f * k2.V + 1.2f * k3.V, y.V), fmaf(ht, 0.3f * k1.w - 0.9f * k2.w + 1.2f * k3.w, y.w), gx_, gi_); }
        { NG_G(fmaf(x, fmaf(x, fmaf(x, fmaf(0.07f, x, 7.f / 60.f), 0.5f), 1.f), 1.f), fmaf(x, fmaf(x, fmaf(0.28f, x, 0.35f), 1.f), 1.f))
#define E5(c) ((-11.f / 54.f) * k1.c + 2.5f * k2.c - (70.f / 27.f) * k3.c + (35.f / 27.f) * k4.c)
          k5 = adex_rhs_vw(p, fmaf(ht, E5(V), y.V), fmaf(ht, E5(w), y.w), gx_, gi_); }
        { NG_G(fmaf(x, fmaf(x, fmaf(x, fmaf(x, fmaf(1771.f / 409600.f, x, 1771.f / 61440.f), 161.f / 1536.f), 49.f / 128.f), 0.875f), 1.f),
               fmaf(x, fmaf(x, fmaf(x, fmaf(1771.f / 81920.f, x, 1771.f / 15360.f), 161.f / 512.f), 49.f / 64.f), 0.875f))
#define E6(c) ((1631.f / 55296.f) * k1.c + (175.f / 512.f) * k2.c + (575.f / 13824.f) * k3.c + (44275.f / 110592.f) * k4.c + (253.f / 4096.f) * k5.c)
          k6 = adex_rhs_vw(p, fmaf(ht, E6(V), y.V), fmaf(ht, E6(w), y.w), gx_, gi_); }
        // 5th-order weights and the difference to the embedded 4th-order ones
#define Y5(c) ((37.f / 378.f) * k1.c + (250.f / 621.f) * k3.c + (125.f / 594.f) * k4.c + (512.f / 1771.f) * k6.c)
#define ER(c) ((37.f / 378.f - 2825.f / 27648.f) * k1.c + (250.f / 621.f - 18575.f / 48384.f) * k3.c + \
               (125.f / 594.f - 13525.f / 55296.f) * k4.c - (277.f / 14336.f) * k5.c + (512.f / 1771.f - 0.25f) * k6.c)
        // error polynomial of the linear pair: e(x) = x^5 (-277/1228800 + 277/1638400 x), h e'(x) likewise
        const float x2 = x * x, x4 = x2 * x2;
        const float eP = x4 * x * fmaf(277.f / 1638400.f, x, -277.f / 1228800.f);
        const float hdE = ht * x4 * fmaf(831.f / 819200.f, x, -277.f / 245760.f);
        float e = fabsf(ht * ER(V)) * p.inv_tol[0];
        e = fmaxf(e, fabsf(ht * ER(w)) * p.inv_tol[1]);
        e = fmaxf(e, fabsf(fmaf(eP, y.gx, hdE * y.yx)) * p.inv_tol[2]);
        e = fmaxf(e, fabsf(eP * y.yx) * p.inv_tol[3]);
        e = fmaxf(e, fabsf(fmaf(eP, y.gi, hdE * y.yi)) * p.inv_tol[4]);
        e = fmaxf(e, fabsf(eP * y.yi) * p.inv_tol[5]);
        const bool accept = e <= 1.f || ht <= p.h_min;
        float fac = e > 0.f ? 0.9f * __powf(e, -0.2f) : 5.f;
        fac = fminf(5.f, fmaxf(0.2f, fac));
        if (!clipped || !accept) h_int = fminf(h_step, ht * fac);
        if (accept) {
            // p(x) = 1 + x + x^2/2 + x^3/6 + x^4/24 + x^5/120 + x^6/800 and h p'(x)
            const float P = fmaf(x, fmaf(x, fmaf(x, fmaf(x, fmaf(x, fmaf(1.f / 800.f, x, 1.f / 120.f), 1.f / 24.f), 1.f / 6.f), 0.5f), 1.f), 1.f);
            const float hdP = ht * fmaf(x, fmaf(x, fmaf(x, fmaf(x, fmaf(3.f / 400.f, x, 1.f / 24.f), 1.f / 6.f), 0.5f), 1.f), 1.f);
            y.V = fmaf(ht, Y5(V), y.V);
            y.w = fmaf(ht, Y5(w), y.w);
            y.gx = fmaf(P, y.gx, hdP * y.yx); y.yx = P * y.yx;
            y.gi = fmaf(P, y.gi, hdP * y.yi); y.yi = P * y.yi;
            t = clipped ? h_step : t + ht;
            if (y.V >= p.V_peak) { y.V = p.V_reset; y.w += p.b; spiked = true; }     // C24; a 2nd crossing is not recorded (C20)
        }
#undef NG_G
#undef E5
#undef E6
#undef Y5
#undef ER
    }
    return true;
}
__device__ __forceinline__ bool adex_step(const AdexDev& p, AdexY& y, float& h_int, float h_step) {
    float t = 0.f;
    bool spiked = false;
    adex_advance<false>(p, y, h_int, t, spiked, h_step);
    return spiked;
}

// kAdex: the network holds AdEx populations (second receptor port, AdEx state arrays); LIF-only networks compile to
// exactly the code without it.
// neuron_load: every load of one neuron-step, issued together (one memory round trip).  Networks that need several
// rounds per step (config 4) issue the loads of the next round before they compute the current one.
struct NeuronLoad { float in, in1, V, I; int r, pi, kq; };

template <bool kAdex>
__device__ __forceinline__ NeuronLoad neuron_load(const StepArgs& a, const float* __restrict__ plane, int i, bool have_k) {
    NeuronLoad L;
    L.in = ld_plane(plane + i);                  // written by red.global from other SMs: read at L2
    L.in1 = kAdex ? ld_plane(plane + a.N + i) : 0.f;          // inhibitory port
    L.kq = have_k ? (int)a.pois_k[i] : 0xff;
    L.V = 0.f; L.I = 0.f; L.r = 0; L.pi = 0;
    if (!a.bypass) { L.V = a.V[i]; L.I = a.I[i]; L.r = a.refr[i]; L.pi = a.pop_of[i]; }
    return L;
}

template <bool kAdex, bool kOneAttempt = false>
__device__ __forceinline__ bool neuron_early(const StepArgs& a, const PopDev* __restrict__ P, long long n, int i,
                                             NeuronRegs& g, const NeuronLoad& L) {
    g.in = L.in; g.in1 = L.in1; g.kq = L.kq; g.adex = false; g.pending = false;
    if (a.bypass) {                                          // DESIGN.md C8: delivery-only mode
        const uint4 x = philox4x32_10(a.seed_lo, a.seed_hi, (uint32_t)(a.id_first + i), (uint32_t)n, (uint32_t)(n >> 32), kTagInject);
        return x.x < a.inject_thr;
    }
    float V = L.V;
    g.I = L.I;
    int r = L.r;
    g.pi = L.pi;
    const PopDev* __restrict__ p = P + g.pi;
    if (kAdex && p->model == 1) {                // AdEx: the whole step is integrated here; neuron_late applies the jumps
        g.adex = true;
        AdexY y; y.V = V; y.w = a.ax_w[i]; y.gx = a.ax_gx[i]; y.yx = a.ax_yx[i]; y.gi = a.ax_gi[i]; y.yi = a.ax_yi[i];
        float h_int = a.ax_h[i];
        g.t = 0.f; g.spiked = false;
        const bool done = adex_advance<kOneAttempt>(p->ax, y, h_int, g.t, g.spiked, a.dt_ms);
        a.V[i] = y.V; a.ax_w[i] = y.w; a.ax_gx[i] = y.gx; a.ax_gi[i] = y.gi; a.ax_h[i] = h_int;
        if (!done) { a.ax_yx[i] = y.yx; a.ax_yi[i] = y.yi; g.pending = true; return false; }    // resumed by adex_resume
        g.I = y.yx;
        a.ax_yi[i] = fmaf(p->ax.jump, g.in1, y.yi);          // C25: jumps arriving at t_{n+1}
        return g.spiked;
    }
    const float E_L = p->E_L;
    bool spk = false;
    if (r == 0) V = E_L + fmaf(p->P22, V - E_L, fmaf(p->P21, g.I, p->P20Ie));
    else r -= 1;
    if (V >= p->V_th) { spk = true; V = p->V_reset; r = p->refr_steps; }
    a.V[i] = V; a.refr[i] = r;
    return spk;
}

template <bool kAdex>
__device__ __forceinline__ void neuron_late(const StepArgs& a, const PopDev* __restrict__ P, long long n, int i,
                                            float* __restrict__ plane, const NeuronRegs& g) {
    clear_plane(plane + i);
    if (kAdex) clear_plane(plane + a.N + i);
    if (a.last_input) { a.last_input[i] = g.in; if (kAdex) a.last_input[a.N + i] = g.in1; }
    if (a.bypass) return;
    const PopDev* __restrict__ p = P + g.pi;
    const int k = g.kq != 0xff ? g.kq : poisson_count(a, p, n, a.id_first + i);
    if (kAdex && g.adex) {                       // g.I carries y_ex after the integration; Poisson drive on the excitatory port
        a.ax_yx[i] = fmaf(p->ax.jump, fmaf(p->w_ext, (float)k, g.in), g.I);
        return;
    }
    a.I[i] = fmaf(p->P11, g.I, g.in) + p->w_ext * (float)k;
}

// Second pass of an AdEx neuron whose first attempt did not complete the step: reload, finish the step, apply the
// conductance jumps and clear the input cells (what neuron_early / neuron_late do for the others).  Returns the spike.
__device__ __noinline__ bool adex_resume(const StepArgs& a, const PopDev* __restrict__ P, long long n, int i, float t, bool spiked,
                                            float* __restrict__ plane) {
    const PopDev* __restrict__ p = P + a.pop_of[i];
    AdexY y; y.V = a.V[i]; y.w = a.ax_w[i]; y.gx = a.ax_gx[i]; y.yx = a.ax_yx[i]; y.gi = a.ax_gi[i]; y.yi = a.ax_yi[i];
    float h_int = a.ax_h[i];
    const float in = ld_plane(plane + i), in1 = ld_plane(plane + a.N + i);
    adex_advance<false>(p->ax, y, h_int, t, spiked, a.dt_ms);
    const int k = poisson_count(a, p, n, a.id_first + i);
    a.V[i] = y.V; a.ax_w[i] = y.w; a.ax_gx[i] = y.gx; a.ax_gi[i] = y.gi; a.ax_h[i] = h_int;
    a.ax_yx[i] = fmaf(p->ax.jump, fmaf(p->w_ext, (float)k, in), y.yx);       // C25
    a.ax_yi[i] = fmaf(p->ax.jump, in1, y.yi);
    clear_plane(plane + i); clear_plane(plane + a.N + i);
    if (a.last_input) { a.last_input[i] = in; a.last_input[a.N + i] = in1; }
    return spiked;
}

template <bool kAdex>
__device__ __forceinline__ void update_phase(const StepArgs& a, const PopDev* __restrict__ P, long long n, int slot,
                                             unsigned long long rec_base, long long gtid, long long gthreads,
                                             unsigned long long win_base = 0) {
    const int N = a.N;
    float* __restrict__ plane = a.ring + (size_t)slot * a.NR;
    const long long n_round = ((long long)N + 31) & ~31LL;      // keep warps whole for the ballot
    for (long long ii = gtid; ii < n_round; ii += gthreads) {
        const int i = (int)ii;
        NeuronRegs g;
        NeuronLoad L;
        if (i < N) L = neuron_load<kAdex>(a, plane, i, false);
        const bool spk = i < N && neuron_early<kAdex>(a, P, n, i, g, L);
        append_spike(a, spk, i, n, rec_base, win_base);
        if (i < N) neuron_late<kAdex>(a, P, n, i, plane, g);
    }
}

// Step bookkeeping of the stand-alone delivery kernels (a4), one thread: publish the next step index, clear the
// spike counter of the next step and advance the record cursor.  (The spike record itself is written by
// append_spike.)  Per-step scalars are always read by ONE thread per CTA and broadcast through shared memory:
// thousands of warps asking the same L2 sector after a barrier serialise on that slice for microseconds.
__device__ __forceinline__ void bookkeeping_scalar(const StepArgs& a, long long n, int slot, int M, unsigned long long rec_base) {
    a.ctl->rec_total[(n + 1) & 1] = rec_base + (unsigned long long)M;
    a.ctl->spike_cnt[(n + 1) & 3] = 0;
    a.ctl->spikes += (unsigned long long)M;
    a.ctl->slot = slot + 1 == a.Dr ? 0 : slot + 1;
    a.ctl->step_u = n + 1;
}

__device__ __forceinline__ void trace_stamp(const StepArgs& a, long long n, int k, int who = 0) {
    if (a.trace && (int)threadIdx.x == who) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        a.trace[((size_t)(n % kTraceSteps) * gridDim.x + blockIdx.x) * kTraceStamps + k] = t;
    }
}
// ---------------------------------------------------------------------------------------
// a3. Spike delivery, kernel 1: row-chunk walk.
//   The CTA stages the spike array's entries (row start, out-degree, padded length — written by append_spike) in
//   shared memory, tile by tile, and prefix-sums their chunk counts; the flattened list of
//   (spike, chunk of kChunkRecords records) items is then dealt round-robin to all warps of the grid: exactly the
//   existing chunks, no per-warp header loads from global memory.  Lane l reads records [4l, 4l+4) of its chunk
//   with one 128-bit load of targets, one of weights and one 32-bit load of delays, then issues up to four
//   red.global.add.f32 into ring[(n + d) mod Dr][target].  Rows are delay-grouped, so consecutive
//   records mostly hit the same ring plane.
// ---------------------------------------------------------------------------------------
constexpr int kEntryTile = 256;
struct DeliverShared {
    long long r0[kEntryTile];
    int32_t len[kEntryTile];
    int32_t pre[kEntryTile + 1];       // pre[k] = chunks of entries [0, k) of the tile
    int32_t warp_tot[kEntryTile / 32];
    int32_t M;
};

// One item: `kPerLane` records per lane (4: 128-bit loads, 1: 32-bit loads) starting at record q of a row.
// A scattered red (or store) instruction holds its warp for about one L2 round trip (~0.45 us measured on B200
// with a quiet memory system), so in the latency regime an item is 32 records — one red per warp — and the
// items are spread over every warp of the grid; under load 128-record items keep the loads 128-bit wide.
template <int kPerLane>
__device__ __forceinline__ void deliver_item(const StepArgs& a, int nmod, long long r0, int len, int c, int lane, int skip = 0) {
    const int Dr = a.Dr;
    const int q = (c * 32 + lane) * kPerLane;
    if (q >= len || q + kPerLane <= skip) return;          // records [0, skip) were delivered by the delay-1 pass
    const long long p = r0 + q;
    int s;
    if (kPerLane == 4) {
        const int4 t = ld_stream_s32x4(a.tgt + p);
        const float4 ww = ld_stream_f32x4(a.w + p);
        const uint32_t dd = ld_stream_u32(a.dly + p);
        if (t.x >= 0 && q >= skip) { s = nmod + (int)(dd & 0xff); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * a.NR + t.x, ww.x); }
        if (t.y >= 0 && q + 1 >= skip) { s = nmod + (int)((dd >> 8) & 0xff); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * a.NR + t.y, ww.y); }
        if (t.z >= 0 && q + 2 >= skip) { s = nmod + (int)((dd >> 16) & 0xff); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * a.NR + t.z, ww.z); }
        if (t.w >= 0 && q + 3 >= skip) { s = nmod + (int)(dd >> 24); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * a.NR + t.w, ww.w); }
    } else if (kPerLane == 2) {
        int2 t; float2 ww; uint32_t dd;
        asm("ld.global.nc.L1::no_allocate.v2.s32 {%0,%1}, [%2];" : "=r"(t.x), "=r"(t.y) : "l"(a.tgt + p));
        asm("ld.global.nc.L1::no_allocate.v2.f32 {%0,%1}, [%2];" : "=f"(ww.x), "=f"(ww.y) : "l"(a.w + p));
        asm("ld.global.nc.L1::no_allocate.u16 %0, [%1];" : "=r"(dd) : "l"(a.dly + p));
        if (t.x >= 0 && q >= skip) { s = nmod + (int)(dd & 0xff); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * a.NR + t.x, ww.x); }
        if (t.y >= 0 && q + 1 >= skip) { s = nmod + (int)(dd >> 8); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * a.NR + t.y, ww.y); }
    } else {
        int t; float ww; uint32_t dd;
        asm("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(t) : "l"(a.tgt + p));
        asm("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(ww) : "l"(a.w + p));
        asm("ld.global.nc.L1::no_allocate.u8 %0, [%1];" : "=r"(dd) : "l"(a.dly + p));
        if (t >= 0) { s = nmod + (int)dd; if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * a.NR + t, ww); }
    }
}

// Returns M, the number of spikes of step n.  Thread 0 reads M while the first kEntryTile threads already load the
// first tile of entries speculatively (one L2 round trip instead of two).
__device__ __forceinline__ int deliver_rows_phase(const StepArgs& a, long long n, int nmod, DeliverShared& sh) {
    const int N = a.NS;
    const RowInfo* __restrict__ rows = a.spike_row + (size_t)(n & 1) * N;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpb = blockDim.x >> 5;
    const int gwarp = blockIdx.x * wpb + wib, gwarps = gridDim.x * wpb;
    if (threadIdx.x == 0) sh.M = __ldcg(&a.ctl->spike_cnt[n & 3]);
    int4 e = make_int4(0, 0, 0, 0);
    if (threadIdx.x < kEntryTile && threadIdx.x < N) e = __ldcg(reinterpret_cast<const int4*>(rows + threadIdx.x));
    __syncthreads();
    const int M = sh.M;
    // latency regime: about two 32-record items per warp or fewer
    const bool small = (long long)M * a.mean_row_records <= 64LL * gwarps;
    const int cshift = small ? 5 : 7;
    unsigned long long ev = 0;
    int base_mod = 0;                                          // (flattened index of the tile's first item) mod gw_n
    // Many spikes (>= 8 per CTA): every CTA stages only its own tiles of the spike array and deals their items to its
    // own warps; few spikes: every CTA stages all of them and the items are dealt to all warps of the grid.
    const bool part = M >= 8 * (int)gridDim.x;
    // a CTA's tile holds about M / gridDim entries, so that every CTA has one
    const int tile_len = part ? min(kEntryTile, (M + (int)gridDim.x - 1) / (int)gridDim.x) : kEntryTile;
    const int tile_first = part ? (int)blockIdx.x * tile_len : 0, tile_stride = part ? (int)gridDim.x * tile_len : kEntryTile;
    const int gw = part ? wib : gwarp, gw_n = part ? wpb : gwarps;
    for (int tile0 = tile_first; tile0 < M; tile0 += tile_stride) {
        const int m = min(tile_len, M - tile0);
        if (tile0 > 0) {
            __syncthreads();                                   // previous tile's readers are done
            if (threadIdx.x < m) e = __ldcg(reinterpret_cast<const int4*>(rows + tile0 + threadIdx.x));
        }
        if (threadIdx.x < kEntryTile) {                        // first 8 warps: stage entries, scan chunk counts
            int x = 0;
            if (threadIdx.x < m) {                             // e = r0 (lo, hi), deg, len
                sh.r0[threadIdx.x] = (long long)(((unsigned long long)(uint32_t)e.y << 32) | (uint32_t)e.x);
                const int len = padded_len(e.z);
                sh.len[threadIdx.x] = len;
                x = (len + (1 << cshift) - 1) >> cshift;
                if (blockIdx.x == 0 || part) ev += (unsigned long long)e.z;
            }
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, x, o);
                if (lane >= o) x += y;
            }
            if (lane == 31) sh.warp_tot[wib] = x;
            e.x = x;                                           // inclusive scan inside the warp
        }
        __syncthreads();
        if (threadIdx.x < kEntryTile) {
            int off = 0;
            for (int k = 0; k < wib; ++k) off += sh.warp_tot[k];
            sh.pre[threadIdx.x + 1] = e.x + off;
            if (threadIdx.x == 0) sh.pre[0] = 0;
        }
        __syncthreads();
        const int total = sh.pre[m];
        int first = gw - base_mod;                             // items are numbered across tiles: round-robin deal
        if (first < 0) first += gw_n;
        for (int it = first; it < total; it += gw_n) {
            int sidx = 0;                                      // number of k in [1, m] with pre[k] <= it
            for (int j = 0; j < m; j += 32) {
                const int k = j + lane + 1;
                const int v = k <= m ? sh.pre[k] : 0x7fffffff;
                sidx += __popc(__ballot_sync(0xffffffffu, v <= it));
            }
            const int c = it - sh.pre[sidx];
            if (small) deliver_item<1>(a, nmod, sh.r0[sidx], sh.len[sidx], c, lane);
            else deliver_item<4>(a, nmod, sh.r0[sidx], sh.len[sidx], c, lane);
        }
        base_mod = (int)(((long long)base_mod + total) % gw_n);
    }
    if (ev) atomicAdd(&a.ctl->events, ev);
    return M;
}

// ---------------------------------------------------------------------------------------
// a3. Spike delivery, kernel 2: delay-major, lane-packed segment walk.
//   work item = (delay d, spike index i), spike fastest, so everything in flight at one time adds into the same one
//   or two ring planes (N*4 bytes each): the reduction target stays L2-resident even when the whole ring
//   (D*N*4 bytes) does not fit, and the delay comes from the group table — a record costs 8 bytes of reads.
//   A warp takes a batch of up to 32 consecutive items: lane l fetches the header of item l (spike id, group
//   bounds, row offset — one latency chain per batch instead of per segment), the segments are cut into 128-bit
//   vectors (4 records, aligned down to the row's 16-byte grid), a warp prefix sum lays all vectors of the batch end
//   to end and every lane finds the segment of its vector by a 5-step shuffle search: lanes stay busy whatever the
//   segment length (1.6 records for out-degree 100, 156 for out-degree 10,000).
//   `batch` shrinks to 1 when there are fewer items than warps, so a quiet step still spreads over the whole grid.
// ---------------------------------------------------------------------------------------
struct VecRef { long long pb; int q, rel_lo, len, slot; bool on; };

// segment of vector v (in the batch-wide numbering) by a 5-step shuffle search over the exclusive prefix `pre`
__device__ __forceinline__ VecRef locate_vec(int v, int total, int pre, long long pbase, int meta, int slot) {
    int k = 0;
#pragma unroll
    for (int st = 16; st > 0; st >>= 1) {
        const int t = __shfl_sync(0xffffffffu, pre, k + st);
        if (t <= v) k += st;
    }
    VecRef r;
    r.pb = __shfl_sync(0xffffffffu, pbase, k);
    const int mt = __shfl_sync(0xffffffffu, meta, k);
    r.slot = __shfl_sync(0xffffffffu, slot, k);
    r.q = (v - __shfl_sync(0xffffffffu, pre, k)) << 2;
    r.rel_lo = mt & 3; r.len = mt >> 2; r.on = v < total;
    return r;
}
__device__ __forceinline__ void red_vec(const StepArgs& a, const VecRef& r, const int4& t, const float4& ww) {
    float* __restrict__ plane = a.ring + (size_t)r.slot * a.NR;
    if (r.q >= r.rel_lo && r.q < r.len) red_add_f32(plane + t.x, ww.x);
    if (r.q + 1 >= r.rel_lo && r.q + 1 < r.len) red_add_f32(plane + t.y, ww.y);
    if (r.q + 2 >= r.rel_lo && r.q + 2 < r.len) red_add_f32(plane + t.z, ww.z);
    if (r.q + 3 >= r.rel_lo && r.q + 3 < r.len) red_add_f32(plane + t.w, ww.w);
}

// kWindow (delivery kernel 4, the paper's spike-buffer mechanism): no ring.  The spikes of the last D steps
// stay in a time-ordered window; a spike of step s "reaches" its connection group of delay d in step n = s + d - 1, so
// the items of step n are (window entry, delay = age + 1) and every reduction goes into the ONE input plane of step n+1.
// `off` (shared memory) holds the W + 1 window offsets of steps n-W+1 .. n and the end.
template <bool kWindow>
__device__ __forceinline__ void deliver_groups_phase(const StepArgs& a, long long n, int nmod, int M, long long gwarp,
                                                     long long gwarps, int lane, const unsigned long long* off = nullptr, int W = 0,
                                                     int age0 = 0) {
    const int N = a.NS, D = a.D, Dr = a.Dr;
    const int32_t* __restrict__ list = a.spike_list + (size_t)(n & 1) * N;
    const long long items = kWindow ? (long long)(off[W] - off[0]) : (long long)M * D;
    if (items == 0) return;
    const long long bsz = (items + gwarps - 1) / gwarps;
    const int batch = bsz > 32 ? 32 : (int)bsz;
    const long long n_batches = (items + batch - 1) / batch;
    const bool small = items < 0x7fffffffLL;                         // 32-bit div/mod is enough (uniform branch)
    unsigned long long ev = 0;

    // Three-stage software pipeline over this warp's batches b, b+gwarps, ...: while batch k is delivered, the group
    // bounds of batch k+1 and the spike ids of batch k+2 are already in flight (the header chain
    // list -> grp_rel/row_off -> records is three dependent DRAM/L2 round trips otherwise paid per batch).
    auto item_of = [&](long long b, int& d, int& si) -> bool {
        const long long it = b * batch + lane;
        if (b >= n_batches || lane >= batch || it >= items) return false;
        if (kWindow) {                                                   // oldest step first: delay-major like the ring walk
            const unsigned long long pos = off[0] + (unsigned long long)it;
            int lo = 0, hi = W;                                          // largest k with off[k] <= pos
            while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (off[mid] <= pos) lo = mid; else hi = mid; }
            d = W - 1 - lo + age0;                                       // 0-based delay index: age of the spike (the newest
                                                                             // staged step has age age0: 0 = the step just updated)
            si = (int)(pos % (unsigned long long)a.win_cap);
        } else if (small) { d = (int)((uint32_t)it / (uint32_t)M); si = (int)((uint32_t)it - (uint32_t)d * (uint32_t)M); }
        else { d = (int)(it / M); si = (int)(it - (long long)d * M); }
        return true;
    };
    auto load_j = [&](long long b) -> int {
        int d, si;
        return item_of(b, d, si) ? __ldcg((kWindow ? a.win_id : list) + si) : -1;
    };
    int d_cur = 0, d_nxt = 0, si_unused;
    uint32_t ga_cur = 0, gb_cur = 0, ga_nxt = 0, gb_nxt = 0;
    long long r0_cur = 0, r0_nxt = 0;
    auto load_g = [&](long long b, int j, int& d, uint32_t& ga, uint32_t& gb, long long& r0) {
        ga = gb = 0; r0 = 0; d = 0;
        if (j >= 0 && item_of(b, d, si_unused)) {
            const uint32_t* __restrict__ g = a.grp_rel + (size_t)j * (D + 1);
            ga = g[d]; gb = g[d + 1];
            r0 = a.row_off[j];
            if (d == age0) ev += g[D];                               // first visit of this spike: count its out-degree once
        }
    };
    long long b = gwarp;
    int j_nxt = load_j(b);
    load_g(b, j_nxt, d_cur, ga_cur, gb_cur, r0_cur);
    j_nxt = load_j(b + gwarps);
    for (; b < n_batches; b += gwarps) {
        load_g(b + gwarps, j_nxt, d_nxt, ga_nxt, gb_nxt, r0_nxt);       // stage B for the next batch
        j_nxt = load_j(b + 2 * gwarps);                                 // stage A for the one after
        // ---- stage C: header of this lane's item of batch b ----
        long long pbase = 0; int rel_lo = 0, len = 0, slot = 0, nvec = 0;
        if (gb_cur > ga_cur) {
            const long long lo = r0_cur + ga_cur;
            pbase = lo & ~3LL;
            rel_lo = (int)(lo - pbase);
            len = rel_lo + (int)(gb_cur - ga_cur);
            nvec = (len + 3) >> 2;
            if (kWindow) slot = nmod == 0 ? 1 : 0;                      // two planes: this step's and the next step's input
            else { slot = nmod + d_cur + 1; if (slot >= Dr) slot -= Dr; }
        }
        int incl = nvec;                                                // lay the vectors of the batch end to end
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        const int pre = incl - nvec;
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        const int meta = (len << 2) | rel_lo;                           // len < 2^29
        for (int base = 0; base < total; base += 64) {                  // two vectors per lane in flight
            const VecRef r0v = locate_vec(base + lane, total, pre, pbase, meta, slot);
            const VecRef r1v = locate_vec(base + 32 + lane, total, pre, pbase, meta, slot);
            int4 t0 = make_int4(0, 0, 0, 0), t1 = t0; float4 w0 = make_float4(0.f, 0.f, 0.f, 0.f), w1 = w0;
            if (r0v.on) { t0 = ld_stream_s32x4(a.tgt + r0v.pb + r0v.q); w0 = ld_stream_f32x4(a.w + r0v.pb + r0v.q); }
            if (r1v.on) { t1 = ld_stream_s32x4(a.tgt + r1v.pb + r1v.q); w1 = ld_stream_f32x4(a.w + r1v.pb + r1v.q); }
            if (r0v.on) red_vec(a, r0v, t0, w0);
            if (r1v.on) red_vec(a, r1v, t1, w1);
        }
        d_cur = d_nxt; ga_cur = ga_nxt; gb_cur = gb_nxt; r0_cur = r0_nxt;
    }
    if (ev) atomicAdd(&a.ctl->events, ev);
}

// ---------------------------------------------------------------------------------------
// a3. Spike delivery, kernel 5: per-delay event queues (two input planes, like kernel 4).
//   For short delay groups (out-degree / D of a few records: config 3 at out-degree 100 and 1000) both the ring walk and the
//   spike-buffer walk read or reduce at random 12-125-byte granularity, and DRAM sectors, not reductions, bound them.  Here a
//   spiking row is read ONCE, whole and coalesced (8 B of target + weight and 1 B of delay per record), at spike time:
//     append (step n):  a CTA flattens the rows of its share of the spike array into batches of kQBatch records, bins a
//                       batch by delay in shared memory, claims a range in the queue of each arrival step n + d with one
//                       atomic per (batch, delay) and stores (target, weight) there in delay-sorted, coalesced runs;
//                       records of delay 1 are reduced straight into the input plane of step n + 1;
//     drain  (step n):  the queue of arrival step n + 1 — complete since the append of step n - 1, because only delays
//                       >= 2 go through a queue — is streamed (8 B per event, 128-bit loads) into the same plane.
//   Both run in the same launch on different CTAs' time lines (odd CTAs append first, even CTAs drain first): the append is
//   DRAM-stream bound (9 B read + 8 B written per event), the drain is bound by the scattered reductions into ONE plane of
//   N * 4 bytes that stays in L2 whatever D is.  Queue of arrival step a = slot a mod D: during step n the appends write
//   every slot except (n + 1) mod D, which is the one being drained; its counter is cleared by the update of step n + 1.
// ---------------------------------------------------------------------------------------
#ifndef NG_Q_THREADS
#define NG_Q_THREADS 256
#endif
constexpr int kQThreads = NG_Q_THREADS;                       // threads per CTA; 1024 / kQThreads CTAs per SM
constexpr int kQVecPerThread = 2;                              // 128-bit vectors (4 records each) per thread and batch
constexpr int kQBatch = kQThreads * kQVecPerThread * 4;        // records per batch
constexpr int kQTailStride = 16;                               // one 128-byte line per queue counter
struct QueueShared {
    long long r0[kEntryTile];
    int32_t pre[kEntryTile + 1];         // 128-bit vectors of the entries [0, k) of the staged tile
    int32_t warp_tot[kEntryTile / 32];
    uint32_t hist[256];                  // records of the batch per delay
    uint32_t sbase[257];                 // exclusive prefix of hist; [D + 1] = records of the batch that go to a queue
    unsigned long long gbase[256];       // start of the range claimed in the queue of that delay's arrival step
    int2 staged[kQBatch];                // the batch in delay order
    uint8_t sbin[kQBatch];               //   and the delay of each staged record
    int32_t nmodD;
};

__device__ __forceinline__ void queue_append_phase(const StepArgs& a, long long n, int M, float* __restrict__ plane1, QueueShared& sh) {
    const int N = a.NS, D = a.D;
    const RowInfo* __restrict__ rows = a.spike_row + (size_t)(n & 1) * N;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int nmodD = sh.nmodD;
    const int tile_len = max(1, min(kEntryTile, (M + (int)gridDim.x - 1) / (int)gridDim.x));
    unsigned long long ev = 0;
    bool overflow = false;
    if (threadIdx.x < 256) sh.hist[threadIdx.x] = 0;
    for (int tile0 = (int)blockIdx.x * tile_len; tile0 < M; tile0 += (int)gridDim.x * tile_len) {
        const int m = min(tile_len, M - tile0);
        __syncthreads();                                       // the previous tile's readers are done
        int x = 0;
        if (threadIdx.x < kEntryTile) {                        // stage the entries, scan their vector counts
            if ((int)threadIdx.x < m) {
                const int4 e = __ldcg(reinterpret_cast<const int4*>(rows + tile0 + threadIdx.x));     // r0 (lo, hi), deg, d1
                sh.r0[threadIdx.x] = (long long)(((unsigned long long)(uint32_t)e.y << 32) | (uint32_t)e.x);
                x = padded_len(e.z) >> 2;
                ev += (unsigned long long)e.z;
            }
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, x, o);
                if (lane >= o) x += y;
            }
            if (lane == 31) sh.warp_tot[wib] = x;
        }
        __syncthreads();
        if (threadIdx.x < kEntryTile) {
            int off = 0;
            for (int k = 0; k < wib; ++k) off += sh.warp_tot[k];
            sh.pre[threadIdx.x + 1] = x + off;
            if (threadIdx.x == 0) sh.pre[0] = 0;
        }
        __syncthreads();
        const int total_vec = sh.pre[m];
        for (int vb = 0; vb < total_vec; vb += kQThreads * kQVecPerThread) {
            int4 t4[kQVecPerThread]; float4 w4[kQVecPerThread]; uint32_t d4[kQVecPerThread];
#pragma unroll
            for (int u = 0; u < kQVecPerThread; ++u) {
                const int v = vb + u * kQThreads + (int)threadIdx.x;
                t4[u] = make_int4(-1, -1, -1, -1); w4[u] = make_float4(0.f, 0.f, 0.f, 0.f); d4[u] = 0;
                if (v < total_vec) {
                    int lo = 0, hi = m;                        // largest e with pre[e] <= v
                    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (sh.pre[mid] <= v) lo = mid; else hi = mid; }
                    const long long p = sh.r0[lo] + ((long long)(v - sh.pre[lo]) << 2);
                    t4[u] = ld_stream_s32x4(a.tgt + p); w4[u] = ld_stream_f32x4(a.w + p); d4[u] = ld_stream_u32(a.dly + p);
                }
            }
            // hist is zero here: cleared before the first batch and in the staging phase of every batch
            uint32_t rank[kQVecPerThread][4];
#pragma unroll
            for (int u = 0; u < kQVecPerThread; ++u) {
                const int tt[4] = {t4[u].x, t4[u].y, t4[u].z, t4[u].w};
                const float ww[4] = {w4[u].x, w4[u].y, w4[u].z, w4[u].w};
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    uint32_t d = tt[c] >= 0 ? (d4[u] >> (8 * c)) & 0xffu : 0u;           // padding records: target -1
                    if (d == 1u) { red_add_f32(plane1 + tt[c], ww[c]); d = 0u; }         // consumed by the very next step
                    d4[u] = (d4[u] & ~(0xffu << (8 * c))) | (d << (8 * c));              // 0 = not queued
#ifdef NG_Q_MATCH
                    const unsigned mask = __match_any_sync(0xffffffffu, d);             // one shared-memory atomic per delay and warp
                    const int leader = __ffs(mask) - 1;
                    uint32_t base = 0;
                    if (d != 0u && lane == leader) base = atomicAdd(&sh.hist[d], (uint32_t)__popc(mask));
                    base = __shfl_sync(0xffffffffu, base, leader);
                    rank[u][c] = base + (uint32_t)__popc(mask & ((1u << lane) - 1u));
#else
                    rank[u][c] = d != 0u ? atomicAdd(&sh.hist[d], 1u) : 0u;             // the order inside a queue is free
#endif
                }
            }
            __syncthreads();                                   // (A) the histogram of the batch is complete
            if (wib == kQThreads / 32 - 1) {                   // the last warp prefix-sums the 256 bins, 8 per lane, while ...
                uint32_t loc[8], sum = 0;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int k = lane * 8 + j;
                    loc[j] = sum;
                    sum += (k >= 2 && k <= D) ? sh.hist[k] : 0u;
                }
                uint32_t incl = sum;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o) incl += y;
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) sh.sbase[lane * 8 + j] = incl - sum + loc[j];
                if (lane == 31) sh.sbase[256] = incl;          // sbase[D + 1] = records of the batch that go to a queue
            }
            for (int k = threadIdx.x; k < 256; k += kQThreads) {   // ... one global atomic per (batch, delay), all in flight together
                const uint32_t h = (k >= 2 && k <= D) ? sh.hist[k] : 0u;
                if (h > 0u) {
                    int qs = nmodD + k; if (qs >= D) qs -= D;  // arrival step n + k
                    sh.gbase[k] = atomicAdd(a.q_tail + (size_t)qs * kQTailStride, (unsigned long long)h);
                }
            }
            __syncthreads();                                   // (B) sbase and gbase are known
            if (threadIdx.x < 256) sh.hist[threadIdx.x] = 0;   // for the next batch
#pragma unroll
            for (int u = 0; u < kQVecPerThread; ++u) {
                const int tt[4] = {t4[u].x, t4[u].y, t4[u].z, t4[u].w};
                const float ww[4] = {w4[u].x, w4[u].y, w4[u].z, w4[u].w};
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const uint32_t d = (d4[u] >> (8 * c)) & 0xffu;
                    if (d != 0u) {
                        const uint32_t pos = sh.sbase[d] + rank[u][c];
                        sh.staged[pos] = make_int2(tt[c], __float_as_int(ww[c]));
                        sh.sbin[pos] = (uint8_t)d;
                    }
                }
            }
            __syncthreads();                                   // (C) the batch is staged in delay order
            const int total = (int)sh.sbase[D + 1];
            for (int p = threadIdx.x; p < total; p += kQThreads) {    // consecutive threads, consecutive queue cells
                const int d = sh.sbin[p];
                int qs = nmodD + d; if (qs >= D) qs -= D;
                const unsigned long long pos = sh.gbase[d] + (unsigned long long)(p - (int)sh.sbase[d]);
                if (pos < (unsigned long long)a.q_cap) a.q_ev[(size_t)qs * (size_t)a.q_cap + pos] = sh.staged[p];
                else overflow = true;
            }
            // no barrier here: the next batch touches only hist before its (A), sbase / gbase after (A), staged after (B)
        }
    }
    if (overflow) a.ctl->err_queue = 1;
    // event counter: one atomic per CTA
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ev += __shfl_xor_sync(0xffffffffu, ev, o);
    __syncthreads();
    if (lane == 0 && wib < kEntryTile / 32) sh.gbase[wib] = ev;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long tot = 0;
        for (int k = 0; k < kEntryTile / 32; ++k) tot += sh.gbase[k];
        if (tot) atomicAdd(&a.ctl->events, tot);
    }
}

__device__ __forceinline__ void queue_drain_phase(const StepArgs& a, float* __restrict__ plane1, const QueueShared& sh) {
    const int D = a.D;
    int qs = sh.nmodD + 1; if (qs >= D) qs -= D;               // arrival step n + 1
    const unsigned long long T0 = __ldcg(a.q_tail + (size_t)qs * kQTailStride);
    const long long T = (long long)(T0 < (unsigned long long)a.q_cap ? T0 : (unsigned long long)a.q_cap);
    const int2* __restrict__ q = a.q_ev + (size_t)qs * (size_t)a.q_cap;
    const long long gtid = (long long)blockIdx.x * blockDim.x + threadIdx.x, gthreads = (long long)gridDim.x * blockDim.x;
    const long long pairs = T >> 1;                            // two events per 128-bit load, four loads in flight per thread
    for (long long i = gtid; i < pairs; i += 4 * gthreads) {
        int4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            v[u] = i + u * gthreads < pairs ? ld_stream_s32x4(reinterpret_cast<const int32_t*>(q + 2 * (i + u * gthreads))) : make_int4(-1, 0, -1, 0);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (v[u].x >= 0) red_add_f32(plane1 + v[u].x, __int_as_float(v[u].y));
            if (v[u].z >= 0) red_add_f32(plane1 + v[u].z, __int_as_float(v[u].w));
        }
    }
    if ((T & 1) && gtid == 0) { const int2 v = q[T - 1]; red_add_f32(plane1 + v.x, __int_as_float(v.y)); }
}

// ---------------------------------------------------------------------------------------
// Population table staged in shared memory (the Poisson CDF walk and the propagators then cost shared-memory
// latency instead of a chain of L2 round trips; L1 is invalidated at every kernel boundary).
// ---------------------------------------------------------------------------------------
constexpr int kMaxPopsSmem = 16;
__device__ __forceinline__ const PopDev* stage_pops(const StepArgs& a, PopDev* sh) {
    if (a.n_pops > kMaxPopsSmem) return a.pops;
    const uint32_t* __restrict__ src = reinterpret_cast<const uint32_t*>(a.pops);
    uint32_t* dst = reinterpret_cast<uint32_t*>(sh);
    const int words = a.n_pops * (int)(sizeof(PopDev) / 4);
    for (int k = threadIdx.x; k < words; k += blockDim.x) dst[k] = __ldg(src + k);
    __syncthreads();
    return sh;
}

// Grid barrier of the persistent kernels: one release-arrival per CTA on a counter that only grows, then an
// acquire-poll by the same thread.  The kernels are launched cooperatively (all CTAs co-resident); the host clears
// ctl->bar before the launch.  Split in two so that work which needs no other CTA's data (the Poisson counts of
// the next step) runs between arrival and release — the ~1 us a barrier costs on this part (one L2 round trip to
// drain the CTA's reductions, one for the arrival, one for the poll) is otherwise idle time.
__device__ __forceinline__ void grid_arrive(Ctl* ctl, unsigned long long& epoch) {
    __syncthreads();
    if (threadIdx.x == 0) {
        epoch += gridDim.x;
        asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(&ctl->bar) : "memory");
    }
}
// Split kernel: a poller that has just seen its barrier incomplete waits a moment before it asks again — hundreds of CTAs
// polling one word back to back queue in front of the arrivals at that word's L2 slice (config 2: 3.73 -> 3.60 us per step with
// 400 cycles, 3.61 with 100, 3.64 with 1000).  Not for grid_wait: where the barrier stands alone between two phases any pause
// is latency (config 0: 2.49 -> 2.67 us with 400 cycles).
#ifndef NG_POLL_PAUSE
#define NG_POLL_PAUSE 400
#endif
__device__ __forceinline__ void poll_pause(int cycles = NG_POLL_PAUSE) {
    const long long c0 = clock64();
    while (clock64() - c0 < cycles) {}
}
__device__ __forceinline__ void grid_wait(Ctl* ctl, unsigned long long epoch) {
    if (threadIdx.x == 0) {
        unsigned long long v;
        do {
            asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(&ctl->bar) : "memory");
        } while (v < epoch);
    }
    __syncthreads();
}
__device__ __forceinline__ void grid_barrier(Ctl* ctl, unsigned long long& epoch) {
    grid_arrive(ctl, epoch);
    grid_wait(ctl, epoch);
}

struct StepScalars { long long n; unsigned long long rec_base; int M; int slot; };
constexpr int kPersistentThreads = 1024;

// ---------------------------------------------------------------------------------------
// Delivery kernel 3: the pipelined step — ONE grid-wide dependency per time step instead of two.
//   Only the delay-1 records of a spike of step n must land before update(n+1) starts; every other record
//   (delay d >= 2, slot n+d) is not consumed before step n+2.  A step is therefore cut differently:
//     phase n = [ update(n), then the CTA delivers the delay-1 records of ITS OWN spikes ]   (critical path)
//               || [ the whole grid delivers the delay >= 2 records of the spikes of step n-1 ] (overlapped)
//     barrier / kernel boundary
//   The delay-1 records are the first RowInfo.d1 records of a row (rows are delay-grouped) —
//   ~140-200 of ~3900 in the microcircuit — so the serial part per spike is one 32-record item per warp.
//   Nothing in a phase reads what the same phase writes: update(n) consumes plane n mod Dr, the delay-1 pass
//   writes plane n+1, the rest pass of step n-1 writes planes n+1 .. n-1+D (Dr = D + 1 planes).
//   The spike record of step n-1 is written by CTA 0 during the rest pass (coalesced, off the critical path).
// ---------------------------------------------------------------------------------------
#ifndef NG_ADEX_REST
#define NG_ADEX_REST 64
#endif
constexpr int kAdexRest = NG_ADEX_REST;   // rest-group threads of the AdEx kernels (the integrator is the step: most warps update)
constexpr int kD1Cap = 256;
constexpr int kResCap = 768;             // updater threads of a 1024-thread CTA at most (pipe_updater_threads)
constexpr int kSlowCap = 512;
struct PipeShared {
    PopDev pops[kMaxPopsSmem];
    DeliverShared d;
    int32_t skip[kEntryTile];
    long long d1_r0[kD1Cap];
    int32_t d1_cnt[kD1Cap];
    int32_t d1_deg[kD1Cap];
    int32_t d1_id[kD1Cap];
    int32_t d1_pre[kD1Cap + 32];
    int32_t slow_id[kSlowCap];             // AdEx neurons whose first integration attempt did not finish the step
    float slow_t[kSlowCap];                //   (bit 30 of the id: already spiked), and the time they reached
    // LIF state of the CTA's neurons, resident for a whole persistent launch when one round of updater threads covers
    // the network (thread t owns neuron blockIdx.x * U + t): read from global memory at entry, written back at exit
    float res_V[kResCap];
    float res_I[kResCap];
    int32_t res_r[kResCap];
    alignas(16) RowInfo res_row[kResCap];
    uint8_t res_pi[kResCap];
    uint8_t res_kq[kResCap];               // Poisson count of the next step (barrier shadow)
    int32_t n_slow;
    int32_t n_d1;
    int32_t n_d1x[2];                      // kEarly: spikes of step m on the CTA list at [m & 1] (counted one phase ahead)
    int32_t phase_cnt[4];                  // split kernel: warp groups of the CTA that are done with the phase of step index s & 3
    StepScalars sc;
    int32_t pending;
    // pipelined spike-buffer backend (kernel 6): absolute window position of the first spike of step s at [s mod (D+1)]
    // for the last D+1 steps, and the staged offsets of the steps whose groups are due in this phase
    unsigned long long wstart[256];
    unsigned long long woff[256];
};

__device__ __forceinline__ void deliver_d1_piece(const StepArgs& a, float* __restrict__ plane1, long long r0, int cnt, int q) {
    if (q < cnt) {
        int t; float ww;
        asm("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(t) : "l"(a.tgt + r0 + q));
        asm("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(ww) : "l"(a.w + r0 + q));
        red_add_f32(plane1 + t, ww);
    }
}

// Warp-specialised: the last `rest_threads` threads of the CTA run the rest pass of step n-1 while the others run
// update(n) and the delay-1 pass, each group synchronising on its own named barrier.
// Returns M_{n-1} (0 if nothing was pending).  `rec_prev` = spikes recorded before step n-1.
__device__ __forceinline__ void group_sync(int id, int count) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
// Delay-1 pass for many spikes per CTA: (spike, record) pairs flattened over the updater threads.
__device__ __noinline__ void d1_flat_pass(const StepArgs& a, PipeShared& sh, float* __restrict__ plane1, int nd1, int U) {
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    if (wib == 0) {
        int carry = 0;
        for (int base = 0; base < nd1; base += 32) {
            int x = base + lane < nd1 ? sh.d1_cnt[base + lane] : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, x, o);
                if (lane >= o) x += y;
            }
            sh.d1_pre[base + lane + 1] = carry + x;
            carry += __shfl_sync(0xffffffffu, x, 31);
        }
        if (lane == 0) sh.d1_pre[0] = 0;
    }
    group_sync(1, U);
    const int T = sh.d1_pre[nd1];
    for (int f = threadIdx.x; f < T; f += U) {
        int lo = 0, hi = nd1;                          // largest s with d1_pre[s] <= f
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (sh.d1_pre[mid] <= f) lo = mid; else hi = mid; }
        deliver_d1_piece(a, plane1, sh.d1_r0[lo], sh.d1_cnt[lo], f - sh.d1_pre[lo]);
    }
}

// item `it` of the staged tile: find its entry (number of k in [1, m] with pre[k] <= it) and deliver its chunk
__device__ __forceinline__ void pipe_one_item(const StepArgs& a, int nmod, PipeShared& sh, int m, int it, int cshift, int lane) {
    int sidx = 0;
    for (int j = 0; j < m; j += 32) {
        const int k = j + lane + 1;
        const int v = k <= m ? sh.d.pre[k] : 0x7fffffff;
        sidx += __popc(__ballot_sync(0xffffffffu, v <= it));
    }
    const int c = it - sh.d.pre[sidx];
    if (cshift == 5) deliver_item<1>(a, nmod, sh.d.r0[sidx], sh.d.len[sidx], c, lane, sh.skip[sidx]);
    else if (cshift == 6) deliver_item<2>(a, nmod, sh.d.r0[sidx], sh.d.len[sidx], c, lane, sh.skip[sidx]);
    else deliver_item<4>(a, nmod, sh.d.r0[sidx], sh.d.len[sidx], c, lane, sh.skip[sidx]);
}
// Updaters per CTA: just enough for one neuron per thread when the network is small enough for a single round
// (every other warp then joins the rest pass), else all but kEntryTile threads.
// AdEx networks spend their step in the integrator: only four warps are set aside for the rest pass there.
__device__ __forceinline__ int pipe_updater_threads(int N, bool heavy_update) {
    const unsigned per_cta = ((unsigned)N + gridDim.x - 1u) / gridDim.x;          // 32-bit: no 64-bit division on the step path
    const int need = (int)((per_cta + 31u) & ~31u);
    const int cap = (int)blockDim.x - (blockDim.x < 512 ? 64 : heavy_update ? kAdexRest : kEntryTile);
    return (int)per_cta <= cap ? max(need, 32) : cap;
}

// kOneRound: one round of updater threads covers the network (the host knows the grid: one neuron per thread).  The
// kernel is then compiled without the multi-round machinery (loads of the next round in flight) and with the row
// descriptor fetched speculatively for every neuron; AdEx networks additionally use the two-pass update: one
// integration attempt per lane, the unfinished neurons in a second, dense pass (10^5 neurons: 33 -> 19 us per step).
// With many rounds per step the update is bound by its memory round trips and the second pass only adds register
// pressure and traffic, so every lane finishes in place there.
// kResM: LIF state resident in (dynamic) shared memory for networks that need SEVERAL rounds of updater threads per step
// (config 4: 10^6 neurons = 9 rounds of 768 threads on 148 CTAs, 13 B per neuron = 90 KB per CTA).  Thread t of CTA b owns
// neurons ((q * gridDim.x + b) * U + t), q = 0..rounds-1, at index q * U + t.  The membrane update and the spike decision
// then read shared memory only; what is left per neuron and step is the input cell (one 4-byte load, four rounds in
// flight, and the store that clears it), issued after the delay-1 records of the CTA's spikes are on their way.
struct ResM { float* V; float* I; int32_t* r; uint8_t* pi; int rounds; };
#ifndef NG_RESM_REST
#define NG_RESM_REST 256
#endif
constexpr int kResMRest = NG_RESM_REST;           // rest-group threads of the kResM kernel

// kEarly (resident LIF state, ring backend): the membrane update of a step needs nothing that the grid barrier in front of
// it publishes — V_{m+1} = f(V_m, I_m), both final in shared memory when the CTA arrives at the barrier of step m - 1;
// only the CURRENT update reads the input cell.  The spike decision of step m is therefore taken between arrival and
// release of barrier m - 1 (resident_decide), where the CTA would only poll: the CTA list of step m is complete and the
// spiking rows are on their way from DRAM when the phase starts, and the phase itself (resident_late) begins with the
// delay-1 reductions.  Arithmetic and order per neuron are those of the in-phase form: bit-identical results.
#ifndef NG_EARLY_POISSON_LATE_U
#define NG_EARLY_POISSON_LATE_U 256      // updater threads per CTA from which the next step's Poisson counts are drawn at the
#endif                                   // end of the phase instead of in the barrier shadow (measured: DESIGN.md section 6)
__device__ __forceinline__ bool resident_decide(const StepArgs& a, const PopDev* __restrict__ P, long long m, PipeShared& sh, int U) {
    const int t = threadIdx.x, lane = t & 31;
    const long long ii = (long long)blockIdx.x * U + t;
    bool spk = false, ovf = false;
    RowInfo r;
    if (ii < a.N) {
        float V = sh.res_V[t];
        int rf = sh.res_r[t];
        const PopDev* __restrict__ p = P + sh.res_pi[t];
        const float E_L = p->E_L;
        if (rf == 0) V = E_L + fmaf(p->P22, V - E_L, fmaf(p->P21, sh.res_I[t], p->P20Ie));
        else rf -= 1;
        if (V >= p->V_th) { spk = true; V = p->V_reset; rf = p->refr_steps; r = sh.res_row[t]; }
        sh.res_V[t] = V; sh.res_r[t] = rf;
    }
    const unsigned mk = __ballot_sync(0xffffffffu, spk);
    if (mk) {                                                  // warp-aggregated append to the CTA's list of step m
        const int leader = __ffs(mk) - 1;
        int lb = 0;
        if (lane == leader) lb = atomicAdd(&sh.n_d1x[m & 1], __popc(mk));
        if (spk && a.prefetch) prefetch_row(a, r);             // delay-1 head first, then the whole row: a barrier ahead of its use
        lb = __shfl_sync(0xffffffffu, lb, leader);
        if (spk) {
            stat_on_spike(a, (int)ii, m);
            const int k = lb + __popc(mk & ((1u << lane) - 1u));
            if (k < kD1Cap) { sh.d1_r0[k] = r.r0; sh.d1_cnt[k] = r.d1; sh.d1_deg[k] = r.deg; sh.d1_id[k] = (int)ii; }
            else ovf = true;                                   // CTA list full: this thread delivers alone in the phase
        }
    }
    return ovf;
}

// Phase n of the updater threads when the spikes of step n were decided ahead (resident_decide): reserve the CTA's slots in
// the global spike array, deliver the delay-1 records, then the current update — the only reader of the input cell.
__device__ __forceinline__ void resident_late(const StepArgs& a, const PopDev* __restrict__ P, long long n, int slot, PipeShared& sh,
                                              int U, bool have_k, bool ovf, bool pois_late) {
    const int N = a.N, Dr = a.Dr, t = threadIdx.x, lane = t & 31, wib = t >> 5, wpu = U >> 5;
    float* __restrict__ plane = a.ring + (size_t)slot * a.NR;
    float* __restrict__ plane1 = a.ring + (size_t)(slot + 1 == Dr ? 0 : slot + 1) * a.NR;
    const long long ii = (long long)blockIdx.x * U + t;
    const int i = (int)ii;
    float res_in = 0.f;
    if (ii < N) res_in = ld_plane(plane + i);                  // first: the one long latency of the phase
    const int nd1 = min(sh.n_d1x[n & 1], kD1Cap);
    if (t == 0) sh.n_d1x[(n + 1) & 1] = 0;                     // last read in phase n - 1; next written after this phase's last barrier
    trace_stamp(a, n, 4);
    int gb = 0;
    if (t == U - 1 && nd1 > 0) gb = atomicAdd(&a.ctl->spike_cnt[n & 3], nd1);
    if (ovf) {
        const RowInfo r = sh.res_row[t];
        for (int q = 0; q < r.d1; ++q) deliver_d1_piece(a, plane1, r.r0, r.d1, q);
        const size_t gk = (size_t)(n & 1) * N + atomicAdd(&a.ctl->spike_cnt[n & 3], 1);
        a.spike_list[gk] = i;
        st_row_info(a.spike_row + gk, r);
    }
    if (nd1 <= 2) {                                            // latency regime: one or two spikes, 32 records per warp
        for (int s = 0; s < nd1; ++s) {
            const long long r0 = sh.d1_r0[s];
            const int cnt = sh.d1_cnt[s];
            for (int q = wib * 32 + lane; q < cnt; q += wpu * 32) deliver_d1_piece(a, plane1, r0, cnt, q);
        }
    } else d1_flat_pass(a, sh, plane1, nd1, U);
    if (ii < N) {                                              // the current update
        const PopDev* __restrict__ p = P + sh.res_pi[t];
        clear_plane(plane + i);
        if (a.last_input) a.last_input[i] = res_in;
        const int k = have_k ? (int)sh.res_kq[t] : poisson_count(a, p, n, i);
        sh.res_I[t] = fmaf(p->P11, sh.res_I[t], res_in) + p->w_ext * (float)k;
    }
    trace_stamp(a, n, 6);
    if (nd1 > 0 && t >= U - 32) {                              // the last updater warp: a2, the global spike array
        gb = __shfl_sync(0xffffffffu, gb, 31);
        for (int s = lane; s < nd1; s += 32) {
            RowInfo r; r.r0 = sh.d1_r0[s]; r.d1 = sh.d1_cnt[s]; r.deg = sh.d1_deg[s];
            const size_t gk = (size_t)(n & 1) * N + gb + s;
            a.spike_list[gk] = sh.d1_id[s];
            st_row_info(a.spike_row + gk, r);
        }
    }
    // Poisson count of step n + 1 (wide CTAs: here, behind the reductions, instead of in front of the barrier poll)
    if (pois_late && ii < N) sh.res_kq[t] = (uint8_t)poisson_count(a, P + sh.res_pi[t], n + 1, i);
}

// kWin (delivery kernel 6, the pipelined spike-buffer backend): two input planes instead of the D + 1 of the ring.  The
// delay-1 pass is unchanged; the rest pass is replaced by the walk over the spike window of the paper's mechanism
// (as in kernel 4): in phase n the rest warps deliver, for every spike of the steps n - D + 1 .. n - 1, the
// connection group whose delay is the spike's age + 1 — everything that arrives in step n + 1 — into the ONE plane of step
// n + 1, which stays in L2 whatever D and the number of receptor ports are.  `wslot` = n mod (D + 1).
template <bool kUpdate, bool kAdex, bool kOneRound = false, bool kRes = false, bool kResM = false, bool kWin = false, bool kEarly = false>
__device__ __forceinline__ int pipelined_phase(const StepArgs& a, const PopDev* __restrict__ P, long long n, int slot, bool pending,
                                               unsigned long long rec_prev, PipeShared& sh, int U, bool have_k = false,
                                               const ResM rm = ResM{}, int wslot = 0, bool ovf = false) {
    static_assert(!kEarly || (kRes && !kWin), "kEarly: resident one-round LIF state on the ring backend");
    const int N = a.N, Dr = a.Dr;
    const int lane = threadIdx.x & 31;
    // U = pipe_updater_threads(N, kAdex), computed once per launch by the caller: its integer division in front of every
    // phase cost all 32 warps ~50 issue slots each, 0.2 us before the first useful instruction
    const int R = blockDim.x - U;                                  // rest group = threads [U, U + R), R >= 64
    const int RT = min(R, kEntryTile);                             // threads of the rest group that stage entries
    const int nmod_prev = slot == 0 ? Dr - 1 : slot - 1;           // (n - 1) mod Dr
    if (threadIdx.x == 0) { sh.n_d1 = 0; sh.n_slow = 0; }
    if (threadIdx.x == U && !pending) sh.d.M = 0;
    __syncthreads();

    if ((int)threadIdx.x < U) {
        // ---- update(n), spike collection, then the delay-1 records of this CTA's spikes ----
        if (kUpdate && kEarly) resident_late(a, P, n, slot, sh, U, have_k, ovf, U >= NG_EARLY_POISSON_LATE_U);
        else if (kUpdate) {
            const int wib = threadIdx.x >> 5, wpu = U >> 5;
            float* __restrict__ plane = a.ring + (size_t)slot * a.NR;
            float* __restrict__ plane1 = a.ring + (size_t)(slot + 1 == Dr ? 0 : slot + 1) * a.NR;
            const bool single_round = kOneRound;
            const long long stride = (long long)gridDim.x * U;
            NeuronLoad L, Ln;
            float res_in = 0.f, res_I = 0.f;
            if (!kAdex && !kRes && !kResM) { const long long i0 = (long long)blockIdx.x * U + threadIdx.x; if (i0 < N) L = neuron_load<kAdex>(a, plane, (int)i0, have_k); }
            int q_idx = threadIdx.x;                               // kResM: index of this thread's neuron of the current round
            for (long long base = (long long)blockIdx.x * U; base < N; base += stride, q_idx += U) {
                const long long ii = base + threadIdx.x;
                const int i = (int)ii;
                NeuronRegs g;
                if (kAdex) {
                    // the state of the next round (ten words per neuron, one 128-byte line per warp and array) is requested
                    // now, so that the round after this one finds it in L1 (state: only this SM touches it) / L2 (input cells)
                    if (lane < 10 && ii - lane + stride < N) {
                        const long long nx = ii - lane + stride;
                        const float* arr = lane == 0 ? a.V : lane == 1 ? a.ax_w : lane == 2 ? a.ax_gx : lane == 3 ? a.ax_yx : lane == 4 ? a.ax_gi
                                           : lane == 5 ? a.ax_yi : lane == 6 ? a.ax_h : lane == 7 ? plane : lane == 8 ? plane + a.N
                                           : reinterpret_cast<const float*>(a.pop_of) - (nx - nx / 4);   // byte array: element nx / 4 of a float view
                        if (lane == 7 || lane == 8) asm volatile("prefetch.global.L2 [%0];" ::"l"(arr + nx));
                        else asm volatile("prefetch.global.L1 [%0];" ::"l"(arr + nx));
                    }
                    if (ii < N) L = neuron_load<kAdex>(a, plane, i, have_k);
                }
                else if (!kOneRound && !kResM && ii + stride < N) Ln = neuron_load<kAdex>(a, plane, (int)(ii + stride), have_k);   // next round's loads in flight
                // the row descriptor is fetched for EVERY neuron together with its state (16 B, L2-resident because it
                // is touched every step): a spiking thread then needs no further memory round trip
                // (only while one round covers the network: for large N the extra 16 B per neuron-step costs more
                // bandwidth than the round trip of the few spiking threads)
                RowInfo r;
                bool spk = false;
                if (kRes) {
                    // Resident LIF state: the membrane update reads nothing but shared memory — V_{n+1} does not depend on
                    // the input arriving in this step — so the spike is known ~0.1 us into the phase and the delay-1
                    // records start at once; the one L2 round trip of the step (the input cell, written by other SMs'
                    // reds) overlaps all of it and is waited for only by the current update at the end.
                    const int t = threadIdx.x;
                    if (ii < N) {
                        res_in = ld_plane(plane + i);                  // first: the one long latency
                        float V = sh.res_V[t];
                        int rf = sh.res_r[t];
                        res_I = sh.res_I[t];
                        const PopDev* __restrict__ p = P + sh.res_pi[t];
                        const float E_L = p->E_L;
                        if (rf == 0) V = E_L + fmaf(p->P22, V - E_L, fmaf(p->P21, res_I, p->P20Ie));
                        else rf -= 1;
                        if (V >= p->V_th) { spk = true; V = p->V_reset; rf = p->refr_steps; r = sh.res_row[t]; }
                        sh.res_V[t] = V; sh.res_r[t] = rf;
                    }
                } else if (kResM) {
                    if (ii < N) {
                        float V = rm.V[q_idx];
                        int rf = rm.r[q_idx];
                        const PopDev* __restrict__ p = P + rm.pi[q_idx];
                        const float E_L = p->E_L;
                        if (rf == 0) V = E_L + fmaf(p->P22, V - E_L, fmaf(p->P21, rm.I[q_idx], p->P20Ie));
                        else rf -= 1;
                        if (V >= p->V_th) { spk = true; V = p->V_reset; rf = p->refr_steps; }
                        rm.V[q_idx] = V; rm.r[q_idx] = rf;
                    }
                } else {
                if (single_round && !kAdex && ii < N) r = ld_row_info(a.row_info + i);     // (AdEx: four registers live across the integrator)
                spk = ii < N && neuron_early<kAdex, kAdex && kOneRound>(a, P, n, i, g, L);
                }
                if (kAdex && kOneRound && ii < N && g.pending) {            // first attempt did not finish: second pass, dense warps
                    const int ks = atomicAdd(&sh.n_slow, 1);
                    if (ks < kSlowCap) { sh.slow_id[ks] = i | (g.spiked ? (1 << 30) : 0); sh.slow_t[ks] = g.t; }
                    else { spk = adex_resume(a, P, n, i, g.t, g.spiked, plane); g.pending = false; g.adex = false; g.pi = -1; }
                }
                if ((!single_round || kAdex) && spk) r = ld_row_info(a.row_info + i);
                const unsigned m = __ballot_sync(0xffffffffu, spk);
                if (m) {                                           // warp-aggregated append to the CTA's own list
                    const int leader = __ffs(m) - 1;
                    int lb = 0;
                    if (lane == leader) lb = atomicAdd(&sh.n_d1, __popc(m));
                    if (spk && a.prefetch && r.d1 > 0) {           // delay-1 head of the row: needed within a microsecond
                        const uint32_t head = (uint32_t)(((long long)r.d1 * 4 + 15) & ~15LL);
                        prefetch_l2_bulk(reinterpret_cast<const char*>(a.tgt + r.r0), head);
                        prefetch_l2_bulk(reinterpret_cast<const char*>(a.w + r.r0), head);
                    }
                    lb = __shfl_sync(0xffffffffu, lb, leader);
                    if (spk) {
                        stat_on_spike(a, i, n);
                        const int k = lb + __popc(m & ((1u << lane) - 1u));
                        if (k < kD1Cap) { sh.d1_r0[k] = r.r0; sh.d1_cnt[k] = r.d1; sh.d1_deg[k] = r.deg; sh.d1_id[k] = i; }
                        else {                                     // CTA list full: this lane does everything alone
                            for (int q = 0; q < r.d1; ++q) deliver_d1_piece(a, plane1, r.r0, r.d1, q);
                            if (a.prefetch && !kWin) prefetch_row(a, r);
                            const size_t gk = (size_t)(n & 1) * N + atomicAdd(&a.ctl->spike_cnt[n & 3], 1);
                            a.spike_list[gk] = i;
                            st_row_info(a.spike_row + gk, r);
                            if (kWin) a.win_id[atomicAdd(&a.ctl->win_tail, 1ULL) % (unsigned long long)a.win_cap] = i;
                        }
                    }
                }
                if (!kRes && !kResM && ii < N && !(kAdex && kOneRound && (g.pending || g.pi < 0))) neuron_late<kAdex>(a, P, n, i, plane, g);
                if (!kAdex && !kOneRound && !kResM) L = Ln;
            }
            if (kAdex && kOneRound) {                               // second pass over the CTA's slow neurons
                group_sync(1, U);
                const int ns = min(sh.n_slow, kSlowCap);
                for (int s = threadIdx.x; s < ns; s += U) {
                    const int e = sh.slow_id[s], i = e & ((1 << 30) - 1);
                    if (adex_resume(a, P, n, i, sh.slow_t[s], (e >> 30) & 1, plane)) {
                        stat_on_spike(a, i, n);
                        const RowInfo r = ld_row_info(a.row_info + i);
                        if (a.prefetch && r.d1 > 0) {
                            const uint32_t head = (uint32_t)(((long long)r.d1 * 4 + 15) & ~15LL);
                            prefetch_l2_bulk(reinterpret_cast<const char*>(a.tgt + r.r0), head);
                            prefetch_l2_bulk(reinterpret_cast<const char*>(a.w + r.r0), head);
                        }
                        const int k = atomicAdd(&sh.n_d1, 1);
                        if (k < kD1Cap) { sh.d1_r0[k] = r.r0; sh.d1_cnt[k] = r.d1; sh.d1_deg[k] = r.deg; sh.d1_id[k] = i; }
                        else {
                            for (int q = 0; q < r.d1; ++q) deliver_d1_piece(a, plane1, r.r0, r.d1, q);
                            if (a.prefetch && !kWin) prefetch_row(a, r);
                            const size_t gk = (size_t)(n & 1) * N + atomicAdd(&a.ctl->spike_cnt[n & 3], 1);
                            a.spike_list[gk] = i;
                            st_row_info(a.spike_row + gk, r);
                            if (kWin) a.win_id[atomicAdd(&a.ctl->win_tail, 1ULL) % (unsigned long long)a.win_cap] = i;
                        }
                    }
                }
            }
            trace_stamp(a, n, 3);
            group_sync(1, U);
            trace_stamp(a, n, 4);
            const int nd1 = min(sh.n_d1, kD1Cap);
            // one atomic per CTA reserves the CTA's slots in the global spike array; its round trip overlaps the
            // delay-1 pass (nothing on the critical path needs the global index)
            // (issued by the LAST updater thread, whose warp has no delay-1 records unless a row has thousands: on the
            // first warps the atomic's round trip was measured in front of the record loads, 0.4 us)
            // The same warp later writes the CTA's entries of the global spike array: no barrier, nothing after the reds
            // on the warps that deliver.
            int gb = 0;
            unsigned long long wp = 0;                             // kWin: the CTA's range in the spike window
            if ((int)threadIdx.x == U - 1 && nd1 > 0) {
                gb = atomicAdd(&a.ctl->spike_cnt[n & 3], nd1);
                if (kWin) wp = atomicAdd(&a.ctl->win_tail, (unsigned long long)nd1);
            }
            // the rest of the spiking rows is read one phase later: request it now, from the LAST updater threads, so
            // that issuing the bulk prefetches overlaps the delay-1 pass of the first warps instead of following it
            if (a.prefetch && !kWin)                                // (window form: the groups are read one per step over D steps)
                for (int s = U - 1 - (int)threadIdx.x; s < nd1; s += U) {
                    RowInfo r; r.r0 = sh.d1_r0[s]; r.d1 = sh.d1_cnt[s]; r.deg = sh.d1_deg[s];
                    prefetch_row(a, r);
                }
            if (nd1 <= 2) {                                        // latency regime: one or two spikes, 32 records per warp
                for (int s = 0; s < nd1; ++s) {
                    const long long r0 = sh.d1_r0[s];
                    const int cnt = sh.d1_cnt[s];
                    for (int q = wib * 32 + lane; q < cnt; q += wpu * 32) deliver_d1_piece(a, plane1, r0, cnt, q);
                }
            } else d1_flat_pass(a, sh, plane1, nd1, U);           // many spikes: out of line, off the latency path
            if (kRes) {                                            // the current update: the only consumer of the input cell
                const long long ii = (long long)blockIdx.x * U + threadIdx.x;
                if (ii < N) {
                    const int t = threadIdx.x, i = (int)ii;
                    const PopDev* __restrict__ p = P + sh.res_pi[t];
                    clear_plane(plane + i);
                    if (a.last_input) a.last_input[i] = res_in;
                    const int k = have_k ? (int)sh.res_kq[t] : poisson_count(a, p, n, i);
                    sh.res_I[t] = fmaf(p->P11, res_I, res_in) + p->w_ext * (float)k;
                }
            }
            if (kResM) {                                           // current update of every round: input cells, four rounds in flight
                for (int q0 = 0; q0 < rm.rounds; q0 += 4) {
                    float inv[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const long long ii = ((long long)(q0 + u) * gridDim.x + blockIdx.x) * U + threadIdx.x;
                        inv[u] = (q0 + u < rm.rounds && ii < N) ? ld_plane(plane + ii) : 0.f;
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const long long ii = ((long long)(q0 + u) * gridDim.x + blockIdx.x) * U + threadIdx.x;
                        if (q0 + u < rm.rounds && ii < N) {
                            const int idx = (q0 + u) * U + threadIdx.x, i = (int)ii;
                            const PopDev* __restrict__ p = P + rm.pi[idx];
                            clear_plane(plane + i);
                            if (a.last_input) a.last_input[i] = inv[u];
                            const int k = poisson_count(a, p, n, i);
                            rm.I[idx] = fmaf(p->P11, rm.I[idx], inv[u]) + p->w_ext * (float)k;
                        }
                    }
                }
            }
            trace_stamp(a, n, 6);
            if (nd1 > 0 && (int)threadIdx.x >= U - 32) {           // the last updater warp (U is a multiple of 32)
                gb = __shfl_sync(0xffffffffu, gb, 31);
                if (kWin) wp = __shfl_sync(0xffffffffu, wp, 31);
                for (int s = lane; s < nd1; s += 32) {             // a2: global spike array; the rest of the row is read
                    RowInfo r; r.r0 = sh.d1_r0[s]; r.d1 = sh.d1_cnt[s]; r.deg = sh.d1_deg[s];       // one phase later
                    const size_t gk = (size_t)(n & 1) * N + gb + s;
                    a.spike_list[gk] = sh.d1_id[s];
                    st_row_info(a.spike_row + gk, r);
                    if (kWin) a.win_id[(wp + (unsigned long long)s) % (unsigned long long)a.win_cap] = sh.d1_id[s];
                }
            }
        }
    } else if (kWin) {
        // ---- window pass: the groups of the spikes of steps n-W .. n-1 that arrive in step n+1 (delay = age + 1 >= 2) ----
        const int t = threadIdx.x - U, wir = t >> 5, wpr = R >> 5, D = a.D, Dp = D + 1;
        const long long np = n - 1;
        if (t == 0) {
            int M = 0;
            if (pending) {                                         // M_{n-1} is final since the barrier: W_n = W_{n-1} + M_{n-1}
                M = __ldcg(&a.ctl->spike_cnt[np & 3]);
                sh.wstart[wslot] = sh.wstart[wslot == 0 ? D : wslot - 1] + (unsigned long long)M;
            }
            sh.d.M = M;
        }
        group_sync(2, R);
        trace_stamp(a, n, 7, U);
        const int M = sh.d.M;
        const int W = (int)(n < (long long)(D - 1) ? n : (long long)(D - 1));
        for (int k = t; k <= W; k += R) { int q = wslot - W + k; if (q < 0) q += Dp; sh.woff[k] = sh.wstart[q]; }
        group_sync(2, R);
        trace_stamp(a, n, 8, U);
        if (blockIdx.x == 0) {
            if (a.rec_cap > 0 && pending) {                        // spike record of step n-1 (coalesced, off the critical path)
                const int32_t* __restrict__ list_prev = a.spike_list + (size_t)(np & 1) * N;
                for (int i = t; i < M; i += R) {
                    const unsigned long long pos = rec_prev + (unsigned long long)i;
                    if (pos < (unsigned long long)a.rec_cap) { a.rec_id[pos] = __ldcg(list_prev + i); a.rec_step[pos] = (int32_t)np; }
                }
            }
            if (t == 0 && sh.woff[W] - sh.woff[0] > (unsigned long long)a.win_cap) a.ctl->err_window = 1;
        }
        deliver_groups_phase<true>(a, n, slot, M, (long long)blockIdx.x * wpr + wir, (long long)gridDim.x * wpr, lane, sh.woff, W, 1);
        trace_stamp(a, n, 9, U);
    } else if (pending) {
        // ---- rest pass of step n-1: records [d1, deg) of every spike ----
        const int t = threadIdx.x - U;                             // index inside the rest group
        const int wir = t >> 5, wpr = R >> 5;
        const long long np = n - 1;
        const RowInfo* __restrict__ rows_prev = a.spike_row + (size_t)(np & 1) * N;
        const int32_t* __restrict__ list_prev = a.spike_list + (size_t)(np & 1) * N;
        const bool rec_cta = blockIdx.x == 0 && a.rec_cap > 0;
        if (t == 0) sh.d.M = __ldcg(&a.ctl->spike_cnt[np & 3]);
        int4 e = make_int4(0, 0, 0, 0);
        int id_prev = 0;
        if (t < RT && t < N) {                                     // speculative: the first tile, before M is known
            e = __ldcg(reinterpret_cast<const int4*>(rows_prev + t));
            if (rec_cta) id_prev = __ldcg(list_prev + t);
        }
        // the first 32 entries go to shared memory before M is known (entries beyond M are stale but valid memory): the
        // barrier that publishes M publishes them too
        if (t < 32 && t < N) {
            sh.d.r0[t] = (long long)(((unsigned long long)(uint32_t)e.y << 32) | (uint32_t)e.x);
            sh.d.len[t] = padded_len(e.z);
            sh.skip[t] = e.w;
        }
        group_sync(2, R);
        trace_stamp(a, n, 7, U);
        const int M = sh.d.M;
        // items are dealt to the rest warps of the grid, CTA by CTA: a light step has fewer items than rest warps, and an SM
        // issues the scattered reductions of its items one address at a time — every SM should get its share
        const int gwarp = wir * gridDim.x + blockIdx.x, gwarps = gridDim.x * wpr;
        // item size: 32 / 64 / 128 records.  A warp's items are serial (every scattered red holds it for an L2 round trip), so
        // small items only while a quarter of the rest warps or fewer get one; beyond that the wide loads of the 128-record
        // item win (measured on config 2 with thresholds 32/64, 16/32, 8/16 per warp: 4.10 / 4.05 / 4.03 us per step)
        const long long est = (long long)M * a.mean_row_records;
        const int cshift = est <= 8LL * gwarps ? 5 : est <= 16LL * gwarps ? 6 : 7;
        unsigned long long ev = 0;
        int base_mod = 0;
        // many spikes (>= 8 per CTA): every CTA stages only its own tiles and deals their items to its own rest warps
        const bool part = M >= 8 * (int)gridDim.x;
        // a CTA's tile holds about M / gridDim entries, so that every CTA has one
        const int tile_len = part ? min(RT, (M + (int)gridDim.x - 1) / (int)gridDim.x) : RT;
        const int tile_first = part ? (int)blockIdx.x * tile_len : 0, tile_stride = part ? (int)gridDim.x * tile_len : RT;
        const int gw = part ? wir : gwarp, gw_n = part ? wpr : gwarps;
        const bool rec_here = a.rec_cap > 0 && (blockIdx.x == 0 || part);
        if (M <= 32) {
            // Latency regime (three steps of four in config 2): no second staging round and no second barrier — every
            // rest warp prefix-sums the chunk counts of the <= 32 entries in its own registers and finds its items by
            // ballot; the first records are requested ~0.5 us earlier.
            const int len_l = lane < M ? sh.d.len[lane] : 0;
            int incl = (len_l + (1 << cshift) - 1) >> cshift;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += y;
            }
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            if (blockIdx.x == 0 && t < M) {                        // warp 0 of CTA 0 still holds the entries: events, spike record
                ev += (unsigned long long)e.z;
                if (rec_cta) {
                    const unsigned long long pos = rec_prev + (unsigned long long)t;
                    if (pos < (unsigned long long)a.rec_cap) { a.rec_id[pos] = id_prev; a.rec_step[pos] = (int32_t)np; }
                }
            }
            for (int it = gwarp; it < total; it += gwarps) {
                const int sidx = __popc(__ballot_sync(0xffffffffu, incl <= it));
                const int before = __shfl_sync(0xffffffffu, incl, sidx > 0 ? sidx - 1 : 0);
                const int c = it - (sidx > 0 ? before : 0);
                if (cshift == 5) deliver_item<1>(a, nmod_prev, sh.d.r0[sidx], sh.d.len[sidx], c, lane, sh.skip[sidx]);
                else if (cshift == 6) deliver_item<2>(a, nmod_prev, sh.d.r0[sidx], sh.d.len[sidx], c, lane, sh.skip[sidx]);
                else deliver_item<4>(a, nmod_prev, sh.d.r0[sidx], sh.d.len[sidx], c, lane, sh.skip[sidx]);
            }
        } else
        for (int tile0 = tile_first; tile0 < M; tile0 += tile_stride) {
            const int m = min(tile_len, M - tile0);
            if (tile0 > 0) {
                group_sync(2, R);
                if (t < m) {
                    e = __ldcg(reinterpret_cast<const int4*>(rows_prev + tile0 + t));
                    if (rec_here) id_prev = __ldcg(list_prev + tile0 + t);
                }
            }
            int x = 0;
            // only the warps that hold entries run the staging code: with all fifteen rest warps in it the few spikes of
            // a latency-bound step cost ~250 issue slots per warp, 0.5 us, before the first record was requested
            const int mw = (m + 31) >> 5;
            if (t < m) {                                           // e = r0 (lo, hi), deg, d1
                const int len = padded_len(e.z);
                sh.d.r0[t] = (long long)(((unsigned long long)(uint32_t)e.y << 32) | (uint32_t)e.x);
                sh.d.len[t] = len;
                sh.skip[t] = e.w;
                x = (len + (1 << cshift) - 1) >> cshift;
                if (blockIdx.x == 0 || part) ev += (unsigned long long)e.z;
                if (rec_here) {
                    const unsigned long long pos = rec_prev + (unsigned long long)(tile0 + t);
                    if (pos < (unsigned long long)a.rec_cap) { a.rec_id[pos] = id_prev; a.rec_step[pos] = (int32_t)np; }
                }
            }
            if (wir < mw) {                                        // whole warps (m <= RT, a multiple of 32)
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int y = __shfl_up_sync(0xffffffffu, x, o);
                    if (lane >= o) x += y;
                }
                if (lane == 31) sh.d.warp_tot[wir] = x;
            }
            if (m > 32) {                                          // several warps hold entries: add the warp offsets
                group_sync(2, R);
                if (wir < mw) {
                    int off = 0;
                    for (int k = 0; k < wir; ++k) off += sh.d.warp_tot[k];
                    sh.d.pre[t + 1] = x + off;
                }
            } else if (t < 32) sh.d.pre[t + 1] = x;                // latency regime: one warp, one barrier
            if (t == 0) sh.d.pre[0] = 0;
            group_sync(2, R);
            trace_stamp(a, n, 8, U);
            const int total = sh.d.pre[m];
            int first = gw - base_mod;                             // items are numbered across tiles: round-robin deal
            if (first < 0) first += gw_n;
            for (int it = first; it < total; it += gw_n) pipe_one_item(a, nmod_prev, sh, m, it, cshift, lane);
            base_mod = (int)(((long long)base_mod + total) % gw_n);
        }
        trace_stamp(a, n, 9, U);
        if (ev) atomicAdd(&a.ctl->events, ev);
    }
    __syncthreads();
    return sh.d.M;
}

// The rest pass of step n - 1 for the split kernel (persistent_split_kernel): the rest group's half of pipelined_phase as
// a function of its own — it is called by the rest group alone, with no CTA-wide barrier around it.  Waits for the list
// barrier of step n - 1 first (`list_need` arrivals on the word of that step's parity).  Returns M_{n-1}.
__device__ __forceinline__ int split_rest_pass(const StepArgs& a, long long n, int slot, unsigned long long rec_prev, PipeShared& sh, int U, int R,
                                               unsigned long long list_need) {
    // U = first thread of the rest group, R = its size
    const int N = a.N, Dr = a.Dr;
    const int lane = threadIdx.x & 31;
    const int RT = min(R, kEntryTile);
    const int nmod_prev = slot == 0 ? Dr - 1 : slot - 1;           // (n - 1) mod Dr
    {
        // ---- rest pass of step n-1: records [d1, deg) of every spike ----
        const int t = threadIdx.x - U;                             // index inside the rest group
        const int wir = t >> 5, wpr = R >> 5;
        const long long np = n - 1;
        constexpr int kListMask = 3;                               // the spike array of four steps is kept
        const RowInfo* __restrict__ rows_prev = a.spike_row + (size_t)(np & kListMask) * N;
        const int32_t* __restrict__ list_prev = a.spike_list + (size_t)(np & kListMask) * N;
        const bool rec_cta = blockIdx.x == 0 && a.rec_cap > 0;
        if (list_need) {                                 // list barrier of step n-1: its spike array is complete
            if (t == 0) {
                unsigned long long v;
                do {
                    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(&a.ctl->bar_list[np & 1].v) : "memory");
                    if (v < list_need) poll_pause();
                } while (v < list_need);
            }
            group_sync(2, R);
        }
        int4 e = make_int4(0, 0, 0, 0);
        int id_prev = 0;
        if (t == 0) sh.d.M = __ldcg(&a.ctl->spike_cnt8[np & 7]);
        if (t < RT && t < N) {                                     // speculative: the first tile, before M is known
            e = __ldcg(reinterpret_cast<const int4*>(rows_prev + t));
            if (rec_cta) id_prev = __ldcg(list_prev + t);
        }
        // the first 32 entries go to shared memory before M is known (entries beyond M are stale but valid memory): the
        // barrier that publishes M publishes them too
        if (t < 32 && t < N) {
            sh.d.r0[t] = (long long)(((unsigned long long)(uint32_t)e.y << 32) | (uint32_t)e.x);
            sh.d.len[t] = padded_len(e.z);
            sh.skip[t] = e.w;
        }
        group_sync(2, R);
        trace_stamp(a, n, 7, U);
        const int M = sh.d.M;
        // items are dealt to the rest warps of the grid, CTA by CTA: a light step has fewer items than rest warps, and an SM
        // issues the scattered reductions of its items one address at a time — every SM should get its share
        const int gwarp = wir * gridDim.x + blockIdx.x, gwarps = gridDim.x * wpr;
        // item size: 32 / 64 / 128 records.  A warp's items are serial (every scattered red holds it for an L2 round trip), so
        // small items only while a quarter of the rest warps or fewer get one; beyond that the wide loads of the 128-record
        // item win (measured on config 2 with thresholds 32/64, 16/32, 8/16 per warp: 4.10 / 4.05 / 4.03 us per step)
        const long long est = (long long)M * a.mean_row_records;
        const int cshift = est <= 8LL * gwarps ? 5 : est <= 16LL * gwarps ? 6 : 7;
        unsigned long long ev = 0;
        int base_mod = 0;
        // many spikes (>= 8 per CTA): every CTA stages only its own tiles and deals their items to its own rest warps
        const bool part = M >= 8 * (int)gridDim.x;
        // a CTA's tile holds about M / gridDim entries, so that every CTA has one
        const int tile_len = part ? min(RT, (M + (int)gridDim.x - 1) / (int)gridDim.x) : RT;
        const int tile_first = part ? (int)blockIdx.x * tile_len : 0, tile_stride = part ? (int)gridDim.x * tile_len : RT;
        const int gw = part ? wir : gwarp, gw_n = part ? wpr : gwarps;
        const bool rec_here = a.rec_cap > 0 && (blockIdx.x == 0 || part);
        if (M <= 32) {
            // Latency regime (three steps of four in config 2): no second staging round and no second barrier — every
            // rest warp prefix-sums the chunk counts of the <= 32 entries in its own registers and finds its items by
            // ballot; the first records are requested ~0.5 us earlier.
            const int len_l = lane < M ? sh.d.len[lane] : 0;
            int incl = (len_l + (1 << cshift) - 1) >> cshift;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += y;
            }
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            if (blockIdx.x == 0 && t < M) {                        // warp 0 of CTA 0 still holds the entries: events, spike record
                ev += (unsigned long long)e.z;
                if (rec_cta) {
                    const unsigned long long pos = rec_prev + (unsigned long long)t;
                    if (pos < (unsigned long long)a.rec_cap) { a.rec_id[pos] = id_prev; a.rec_step[pos] = (int32_t)np; }
                }
            }
            for (int it = gwarp; it < total; it += gwarps) {
                const int sidx = __popc(__ballot_sync(0xffffffffu, incl <= it));
                const int before = __shfl_sync(0xffffffffu, incl, sidx > 0 ? sidx - 1 : 0);
                const int c = it - (sidx > 0 ? before : 0);
                if (cshift == 5) deliver_item<1>(a, nmod_prev, sh.d.r0[sidx], sh.d.len[sidx], c, lane, sh.skip[sidx]);
                else if (cshift == 6) deliver_item<2>(a, nmod_prev, sh.d.r0[sidx], sh.d.len[sidx], c, lane, sh.skip[sidx]);
                else deliver_item<4>(a, nmod_prev, sh.d.r0[sidx], sh.d.len[sidx], c, lane, sh.skip[sidx]);
            }
        } else
        for (int tile0 = tile_first; tile0 < M; tile0 += tile_stride) {
            const int m = min(tile_len, M - tile0);
            if (tile0 > 0) {
                group_sync(2, R);
                if (t < m) {
                    e = __ldcg(reinterpret_cast<const int4*>(rows_prev + tile0 + t));
                    if (rec_here) id_prev = __ldcg(list_prev + tile0 + t);
                }
            }
            int x = 0;
            // only the warps that hold entries run the staging code: with all fifteen rest warps in it the few spikes of
            // a latency-bound step cost ~250 issue slots per warp, 0.5 us, before the first record was requested
            const int mw = (m + 31) >> 5;
            if (t < m) {                                           // e = r0 (lo, hi), deg, d1
                const int len = padded_len(e.z);
                sh.d.r0[t] = (long long)(((unsigned long long)(uint32_t)e.y << 32) | (uint32_t)e.x);
                sh.d.len[t] = len;
                sh.skip[t] = e.w;
                x = (len + (1 << cshift) - 1) >> cshift;
                if (blockIdx.x == 0 || part) ev += (unsigned long long)e.z;
                if (rec_here) {
                    const unsigned long long pos = rec_prev + (unsigned long long)(tile0 + t);
                    if (pos < (unsigned long long)a.rec_cap) { a.rec_id[pos] = id_prev; a.rec_step[pos] = (int32_t)np; }
                }
            }
            if (wir < mw) {                                        // whole warps (m <= RT, a multiple of 32)
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int y = __shfl_up_sync(0xffffffffu, x, o);
                    if (lane >= o) x += y;
                }
                if (lane == 31) sh.d.warp_tot[wir] = x;
            }
            if (m > 32) {                                          // several warps hold entries: add the warp offsets
                group_sync(2, R);
                if (wir < mw) {
                    int off = 0;
                    for (int k = 0; k < wir; ++k) off += sh.d.warp_tot[k];
                    sh.d.pre[t + 1] = x + off;
                }
            } else if (t < 32) sh.d.pre[t + 1] = x;                // latency regime: one warp, one barrier
            if (t == 0) sh.d.pre[0] = 0;
            group_sync(2, R);
            trace_stamp(a, n, 8, U);
            const int total = sh.d.pre[m];
            int first = gw - base_mod;                             // items are numbered across tiles: round-robin deal
            if (first < 0) first += gw_n;
            for (int it = first; it < total; it += gw_n) pipe_one_item(a, nmod_prev, sh, m, it, cshift, lane);
            base_mod = (int)(((long long)base_mod + total) % gw_n);
        }
        trace_stamp(a, n, 9, U);
        if (ev) atomicAdd(&a.ctl->events, ev);
        return M;
    }
}

// Graph / plain-launch form: one launch per time step, the kernel boundary is the barrier.  The last CTA to finish
// publishes the next step index (a4) and marks the rest pass of this step as pending.
constexpr int kPipeThreads = 512;        // 256 updaters + 256 rest-pass threads
template <bool kUpdate, bool kAdex, bool kOneRound = false>
__global__ void __launch_bounds__(kPipeThreads) pipe_step_kernel(const NG_GC StepArgs a) {
    __shared__ PipeShared sh;
    if (threadIdx.x == 0) {
        sh.sc.n = __ldcg(&a.ctl->step_u);
        sh.sc.slot = __ldcg(&a.ctl->slot);
        sh.pending = __ldcg(&a.ctl->pending);
        sh.sc.rec_base = __ldcg(&a.ctl->rec_total[(sh.sc.n - 1) & 1]);     // recorded before step n-1
    }
    const PopDev* P = stage_pops(a, sh.pops);
    if (a.n_pops > kMaxPopsSmem) __syncthreads();
    const long long n = sh.sc.n;
    const int slot = sh.sc.slot;
    pipelined_phase<kUpdate, kAdex, kOneRound>(a, P, n, slot, sh.pending != 0, sh.sc.rec_base, sh, pipe_updater_threads(a.N, kAdex));
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned t = atomicAdd(&a.ctl->ticket, 1u);
        if (t == gridDim.x - 1) {
            __threadfence();
            a.ctl->ticket = 0;
            if (kUpdate) {
                const int M = __ldcg(&a.ctl->spike_cnt[n & 3]);
                a.ctl->rec_total[(n + 1) & 1] = __ldcg(&a.ctl->rec_total[n & 1]) + (unsigned long long)M;
                a.ctl->spike_cnt[(n + 1) & 3] = 0;
                a.ctl->spikes += (unsigned long long)M;
                a.ctl->step_d = n;
                a.ctl->slot = slot + 1 == a.Dr ? 0 : slot + 1;
                a.ctl->step_u = n + 1;
                a.ctl->pending = 1;
            } else a.ctl->pending = 0;                             // flush launch: rest pass of step n-1 done
        }
    }
}

// kAdex: the AdEx integrator needs more than the 64 registers a 1024-thread CTA leaves: 512-thread CTAs, two per SM at most
template <bool kAdex, bool kOneRound = false, bool kResM = false, bool kWin = false, bool kEarly = false>
__global__ void __launch_bounds__(kAdex ? 512 : kPersistentThreads, kAdex ? 2 : 1) persistent_pipe_kernel(const NG_GC StepArgs a, long long n_steps) {
    __shared__ PipeShared sh;
    if (threadIdx.x == 0) {
        sh.sc.n = __ldcg(&a.ctl->step_u);
        sh.sc.slot = __ldcg(&a.ctl->slot);
        sh.sc.rec_base = __ldcg(&a.ctl->rec_total[sh.sc.n & 1]);
        sh.sc.M = kWin ? (int)(sh.sc.n % (a.D + 1)) : 0;           // kWin: window slot of the first step of this launch
    }
    if (kWin)                                                      // window starts of the last D + 1 steps (Ctl.win_start, [s mod (D+1)])
        for (int k = threadIdx.x; k <= a.D; k += blockDim.x) sh.wstart[k] = __ldcg(&a.ctl->win_start[k]);
    const PopDev* P = stage_pops(a, sh.pops);
    if (a.n_pops > kMaxPopsSmem) __syncthreads();
    const long long gtid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int U = kResM ? (int)blockDim.x - kResMRest : pipe_updater_threads(a.N, kAdex);
    const bool single_round = kOneRound;                           // else the counts are computed in line, overlapping the loads
    constexpr bool kRes = !kAdex && kOneRound;                     // LIF state resident in shared memory (the host never
    const long long res_i = (long long)blockIdx.x * U + threadIdx.x;       // picks this instantiation in bypass mode)
    if (kRes && (int)threadIdx.x < U && res_i < a.N) {
        const int t = threadIdx.x;
        sh.res_V[t] = a.V[res_i]; sh.res_I[t] = a.I[res_i]; sh.res_r[t] = a.refr[res_i]; sh.res_pi[t] = a.pop_of[res_i];
        sh.res_row[t] = ld_row_info(a.row_info + res_i);
    }
    ResM rm{};
    if constexpr (kResM) {
        extern __shared__ __align__(16) unsigned char res_dyn[];   // V, I_syn, refr, population byte of the CTA's neurons
        const long long per_round = (long long)gridDim.x * U;
        rm.rounds = (int)((a.N + per_round - 1) / per_round);
        const size_t cap = (size_t)rm.rounds * U;
        rm.V = reinterpret_cast<float*>(res_dyn); rm.I = rm.V + cap;
        rm.r = reinterpret_cast<int32_t*>(rm.I + cap); rm.pi = reinterpret_cast<uint8_t*>(rm.r + cap);
        if ((int)threadIdx.x < U)
            for (int q = 0; q < rm.rounds; ++q) {
                const long long ii = ((long long)q * gridDim.x + blockIdx.x) * U + threadIdx.x;
                if (ii < a.N) { const int k = q * U + threadIdx.x; rm.V[k] = a.V[ii]; rm.I[k] = a.I[ii]; rm.r[k] = a.refr[ii]; rm.pi[k] = a.pop_of[ii]; }
            }
    }
    long long n = sh.sc.n;
    int slot = sh.sc.slot;
    unsigned long long rec_prev = sh.sc.rec_base, spikes = 0, epoch = 0;       // recorded before step n-1 (nothing pending at entry)
    int wslot = sh.sc.M;
    bool ovf = false;                                              // kEarly: this thread's spike of the coming step is not on the CTA list
    if (kEarly && n_steps > 0) {                                   // spikes of the first step of the launch
        if (threadIdx.x < 2) sh.n_d1x[threadIdx.x] = 0;
        __syncthreads();
        if ((int)threadIdx.x < U) ovf = resident_decide(a, P, n, sh, U);
    }
    for (long long s = 0; s < n_steps; ++s, ++n) {
        if (gtid == 0) a.ctl->spike_cnt[(n + 1) & 3] = 0;          // last read (as step n-3's) in phase n-2
        trace_stamp(a, n, 0);
        const int Mp = pipelined_phase<true, kAdex, kOneRound, kRes, kResM, kWin, kEarly>(a, P, n, slot, s > 0, rec_prev, sh, U, s > 0 && single_round, rm, wslot, ovf);
        rec_prev += (unsigned long long)Mp; spikes += (unsigned long long)Mp;
        trace_stamp(a, n, 1);
        grid_arrive(a.ctl, epoch);
        if (s + 1 < n_steps && !a.bypass && single_round && (int)threadIdx.x < U) {    // barrier shadow: Poisson counts of step n+1
            if (kEarly) {                                          // ... and, first, its spikes
                ovf = resident_decide(a, P, n + 1, sh, U);
                const long long ii = (long long)blockIdx.x * U + threadIdx.x;
                if (U < NG_EARLY_POISSON_LATE_U && ii < a.N) sh.res_kq[threadIdx.x] = (uint8_t)poisson_count(a, P + sh.res_pi[threadIdx.x], n + 1, (int)ii);
            } else if (kRes) {                                     // thread t owns neuron blockIdx.x * U + t for the whole launch
                const long long ii = (long long)blockIdx.x * U + threadIdx.x;
                if (ii < a.N) sh.res_kq[threadIdx.x] = (uint8_t)poisson_count(a, P + sh.res_pi[threadIdx.x], n + 1, (int)ii);
            } else
                for (long long ii = (long long)blockIdx.x * U + threadIdx.x; ii < a.N; ii += (long long)gridDim.x * U)
                    a.pois_k[ii] = (uint8_t)poisson_count(a, P + a.pop_of[ii], n + 1, (int)ii);
        }
        grid_wait(a.ctl, epoch);
        trace_stamp(a, n, 2);
        slot = slot + 1 == a.Dr ? 0 : slot + 1;
        if (kWin) wslot = wslot == a.D ? 0 : wslot + 1;
    }
    if (kRes && (int)threadIdx.x < U && res_i < a.N) {
        const int t = threadIdx.x;
        a.V[res_i] = sh.res_V[t]; a.I[res_i] = sh.res_I[t]; a.refr[res_i] = sh.res_r[t];
    }
    if (kResM && (int)threadIdx.x < U)
        for (int q = 0; q < rm.rounds; ++q) {
            const long long ii = ((long long)q * gridDim.x + blockIdx.x) * U + threadIdx.x;
            if (ii < a.N) { const int k = q * U + threadIdx.x; a.V[ii] = rm.V[k]; a.I[ii] = rm.I[k]; a.refr[ii] = rm.r[k]; }
        }
    if (kWin) {
        // nothing to flush: what is still due lives in the spike window and the plane of step n is complete.  Close the
        // bookkeeping of the last step (its count, its window start, its part of the spike record) for the next call.
        if (n_steps > 0) {
            __syncthreads();
            if (threadIdx.x == 0) sh.d.M = __ldcg(&a.ctl->spike_cnt[(n - 1) & 3]);
            __syncthreads();
            const int Ml = sh.d.M;
            if (blockIdx.x == 0) {
                if (threadIdx.x == 0) sh.wstart[wslot] = sh.wstart[wslot == 0 ? a.D : wslot - 1] + (unsigned long long)Ml;
                __syncthreads();
                for (int k = threadIdx.x; k <= a.D; k += blockDim.x) a.ctl->win_start[k] = sh.wstart[k];
                if (a.rec_cap > 0) {
                    const int32_t* __restrict__ list_prev = a.spike_list + (size_t)((n - 1) & 1) * a.NS;
                    for (int i = threadIdx.x; i < Ml; i += blockDim.x) {
                        const unsigned long long pos = rec_prev + (unsigned long long)i;
                        if (pos < (unsigned long long)a.rec_cap) { a.rec_id[pos] = __ldcg(list_prev + i); a.rec_step[pos] = (int32_t)(n - 1); }
                    }
                }
            }
            rec_prev += (unsigned long long)Ml; spikes += (unsigned long long)Ml;
        }
    } else if (n_steps > 0) {                                      // flush: rest pass of the last step
        const int Mp = pipelined_phase<false, kAdex>(a, P, n, slot, true, rec_prev, sh, U);
        rec_prev += (unsigned long long)Mp; spikes += (unsigned long long)Mp;
    }
    if (gtid == 0) {
        a.ctl->rec_total[n & 1] = rec_prev;
        a.ctl->rec_total[(n - 1) & 1] = rec_prev;
        a.ctl->spikes += spikes;
        a.ctl->step_d = n - 1;
        a.ctl->slot = slot;
        a.ctl->step_u = n;
    }
}

// ---------------------------------------------------------------------------------------
// The split kernel: the resident LIF kernel (kEarly) with its grid barrier cut in two and its two warp groups decoupled.
//   What a step really orders across CTAs is two things:
//     list(n):  every CTA has appended its spikes of step n to the global spike array           -> Ctl::bar_list[n & 1]
//     plane(n): every CTA has issued (and had acknowledged) all reductions of phase n           -> Ctl::bar_plane[step index & 1]
//   and each has ONE consumer: the rest pass of step n (the delay >= 2 records, run by the rest warps) needs list(n); the
//   current update of step n + 1 (the only reader of an input cell) needs plane(n).  Nothing else of a phase reads what
//   other CTAs wrote in the phase before — the ring has D + 1 planes, the spike array is kept for four steps and its
//   counters for eight — so no warp waits at a phase boundary any more, and the two warp groups of a CTA run their own loops:
//     updaters, step n:  reserve slots, delay-1 reductions, a2 -> arrive list(n) -> [group done] -> wait plane(n - 1)
//                        -> input cell, current update -> decisions of step n + 1 (resident_decide), its Poisson counts
//     rest warps, step n: wait list(n - 1) -> count, descriptors, records, reductions of step n - 1 -> [group done]
//   The group that is done second in a CTA arrives at plane(n) (one fence each, cumulative over the group's barrier).
//   The latency of a barrier (release fence, arrival, poll: 1.1 us of a 4 us step) then overlaps the other group's work
//   instead of standing between two phases.  Arithmetic and order per neuron are those of the in-phase form.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void split_group_done(const StepArgs& a, PipeShared& sh, long long s_idx) {       // one thread, behind its group's barrier
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
    if (atomicAdd(&sh.phase_cnt[s_idx & 3], 1) == 1) {             // the other group was first: the CTA is done with the phase
        sh.phase_cnt[s_idx & 3] = 0;
        asm volatile("red.relaxed.gpu.global.add.u64 [%0], 1;" ::"l"(&a.ctl->bar_plane[s_idx & 1].v) : "memory");
    }
}

__device__ __forceinline__ bool split_update_step(const StepArgs& a, const PopDev* __restrict__ P, long long n, long long s_idx, int slot,
                                                  PipeShared& sh, int U, bool have_k, bool ovf, unsigned long long plane_need, bool decide_next) {
    const int N = a.N, Dr = a.Dr, t = threadIdx.x, lane = t & 31, wib = t >> 5, wpu = U >> 5;
    float* __restrict__ plane = a.ring + (size_t)slot * a.NR;
    float* __restrict__ plane1 = a.ring + (size_t)(slot + 1 == Dr ? 0 : slot + 1) * a.NR;
    const size_t buf = (size_t)(n & 3) * N;                    // the spike array of step n
    const long long ii = (long long)blockIdx.x * U + t;
    const int i = (int)ii;
    group_sync(1, U);                                          // the CTA list of step n (resident_decide) is complete
    const int n_all = sh.n_d1x[n & 1], nd1 = min(n_all, kD1Cap);
    trace_stamp(a, n, 0);
    // thread 0 asks for plane(n - 1) at once: its round trip runs beside the reductions and the append of the other warps
    if (t == 0 && plane_need) {
        unsigned long long v;
        do {
            asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(&a.ctl->bar_plane[(s_idx - 1) & 1].v) : "memory");
            if (v < plane_need) poll_pause();
        } while (v < plane_need);
    }
    int gb = 0;
    if (t == U - 1 && nd1 > 0) gb = atomicAdd(&a.ctl->spike_cnt8[n & 7], nd1);
    if (ovf) {
        const RowInfo r = sh.res_row[t];
        for (int q = 0; q < r.d1; ++q) deliver_d1_piece(a, plane1, r.r0, r.d1, q);
        const size_t gk = buf + atomicAdd(&a.ctl->spike_cnt8[n & 7], 1);
        a.spike_list[gk] = i;
        st_row_info(a.spike_row + gk, r);
    }
    if (nd1 <= 2) {                                            // latency regime: one or two spikes, 32 records per warp
        for (int s = 0; s < nd1; ++s) {
            const long long r0 = sh.d1_r0[s];
            const int cnt = sh.d1_cnt[s];
            for (int q = wib * 32 + lane; q < cnt; q += wpu * 32) deliver_d1_piece(a, plane1, r0, cnt, q);
        }
    } else d1_flat_pass(a, sh, plane1, nd1, U);
    if (n_all > kD1Cap) group_sync(1, U);                      // overflow lanes have appended alone: before the list arrival
    if (t >= U - 32) {                                         // the last updater warp: a2, the global spike array, list arrival
        gb = __shfl_sync(0xffffffffu, gb, 31);
        for (int s = lane; s < nd1; s += 32) {
            RowInfo r; r.r0 = sh.d1_r0[s]; r.d1 = sh.d1_cnt[s]; r.deg = sh.d1_deg[s];
            a.spike_list[buf + gb + s] = sh.d1_id[s];
            st_row_info(a.spike_row + buf + gb + s, r);
        }
        __syncwarp();
        if (lane == 31) asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(&a.ctl->bar_list[n & 1].v) : "memory");
    }
    // beside those round trips: the Poisson count of step n + 1 (a pure function of neuron and step; 0.85 us for 17 warps)
    int k_cur = -1;
    if (ii < N) {
        if (have_k) k_cur = (int)sh.res_kq[t];
        if (decide_next) sh.res_kq[t] = (uint8_t)poisson_count(a, P + sh.res_pi[t], n + 1, i);
    }
    group_sync(1, U);                                          // all reductions of the phase issued; plane(n - 1) is complete
    trace_stamp(a, n, 4);
    float res_in = 0.f;
    if (ii < N) res_in = ld_plane(plane + i);
    if (t == (U >= 64 ? 32 : 0)) split_group_done(a, sh, s_idx);   // (behind the load: the fence waits for it anyway; measured best place)
    if (t == 0) {
        sh.n_d1x[(n + 1) & 1] = 0;                             // (read above by every warp; written again behind the barrier below)
        // every CTA is done with phase n - 1, hence with the count of step n - 3 (read by the rest pass of phase n - 2):
        // that counter serves step n + 5 next
        if (blockIdx.x == 0) a.ctl->spike_cnt8[(n + 5) & 7] = 0;
    }
    if (ii < N) {                                              // the current update
        const PopDev* __restrict__ p = P + sh.res_pi[t];
        clear_plane(plane + i);
        if (a.last_input) a.last_input[i] = res_in;
        const int k = k_cur >= 0 ? k_cur : poisson_count(a, p, n, i);
        sh.res_I[t] = fmaf(p->P11, sh.res_I[t], res_in) + p->w_ext * (float)k;
    }
    trace_stamp(a, n, 6);
    bool ovf_next = false;
    if (decide_next) {
        group_sync(1, U);                                      // the counter of the next CTA list is clear
        ovf_next = resident_decide(a, P, n + 1, sh, U);
    }
    trace_stamp(a, n, 1);
    return ovf_next;
}

__global__ void __launch_bounds__(kPersistentThreads, 1) persistent_split_kernel(const NG_GC StepArgs a, long long n_steps) {
    __shared__ PipeShared sh;
    if (threadIdx.x == 0) {
        sh.sc.n = __ldcg(&a.ctl->step_u);
        sh.sc.slot = __ldcg(&a.ctl->slot);
        sh.sc.rec_base = __ldcg(&a.ctl->rec_total[sh.sc.n & 1]);
    }
    if (threadIdx.x < 4) sh.phase_cnt[threadIdx.x] = 0;
    if (threadIdx.x < 2) sh.n_d1x[threadIdx.x] = 0;
    const PopDev* P = stage_pops(a, sh.pops);
    __syncthreads();
    const long long gtid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int U = pipe_updater_threads(a.N, false), R = (int)blockDim.x - U;
    const long long res_i = (long long)blockIdx.x * U + threadIdx.x;
    const bool updater = (int)threadIdx.x < U;
    if (updater && res_i < a.N) {
        const int t = threadIdx.x;
        sh.res_V[t] = a.V[res_i]; sh.res_I[t] = a.I[res_i]; sh.res_r[t] = a.refr[res_i]; sh.res_pi[t] = a.pop_of[res_i];
        sh.res_row[t] = ld_row_info(a.row_info + res_i);
    }
    const long long n0 = sh.sc.n;
    const int slot0 = sh.sc.slot;
    unsigned long long rec_prev = sh.sc.rec_base, spikes = 0, epoch = 0;
    bool ovf = false;
    if (n_steps > 0) {
        if (gtid < 5) a.ctl->spike_cnt8[(n0 + gtid) & 7] = 0;      // (the updaters clear the counter of the fifth step ahead)
        if (updater) ovf = resident_decide(a, P, n0, sh, U);       // spikes of the first step of the launch
        grid_barrier(a.ctl, epoch);                                // the counters are clear before any CTA appends
    }
    const unsigned long long G = gridDim.x;
    long long n = n0;
    int slot = slot0;
    int M_last = 0;
    if (updater) {
        for (long long s = 0; s < n_steps; ++s, ++n) {
            // plane(step index s - 1) is the ((s - 1) / 2 + 1)-th use of its word
            ovf = split_update_step(a, P, n, s, slot, sh, U, s > 0, ovf, s > 0 ? (unsigned long long)(((s - 1) >> 1) + 1) * G : 0ULL, s + 1 < n_steps);
            slot = slot + 1 == a.Dr ? 0 : slot + 1;
        }
    } else {
        // ---- the rest warps: list(n - 1), then count, descriptors, records and reductions of step n - 1, then the group's arrival ----
        const int t = threadIdx.x - U;
        for (long long s = 0; s < n_steps; ++s, ++n) {
            if (s > 0) {
                const int Mp = split_rest_pass(a, n, slot, rec_prev, sh, U, R, (unsigned long long)((s + 1) >> 1) * G);
                rec_prev += (unsigned long long)Mp; spikes += (unsigned long long)Mp;
            }
            group_sync(2, R);                                      // every rest warp has issued its reductions of this phase
            if (t == 0) split_group_done(a, sh, s);
            slot = slot + 1 == a.Dr ? 0 : slot + 1;
        }
    }
    // the one full stop of the launch: plane(last step)
    __syncthreads();
    if (n_steps > 0) {
        if (threadIdx.x == 0) {
            unsigned long long v;
            do {
                asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(&a.ctl->bar_plane[(n_steps - 1) & 1].v) : "memory");
            } while (v < (unsigned long long)(((n_steps - 1) >> 1) + 1) * G);
        }
        __syncthreads();
    }
    if (updater && res_i < a.N) {
        const int t = threadIdx.x;
        a.V[res_i] = sh.res_V[t]; a.I[res_i] = sh.res_I[t]; a.refr[res_i] = sh.res_r[t];
    }
    if (n_steps > 0 && !updater) {                                 // flush: rest pass of the last step
        M_last = split_rest_pass(a, n, slot, rec_prev, sh, U, R, (unsigned long long)((n_steps + 1) >> 1) * G);
        rec_prev += (unsigned long long)M_last; spikes += (unsigned long long)M_last;
        if (blockIdx.x == 0) {
            group_sync(2, R);
            if (((n - 1) & 3) >= 2) {                              // the host reads the last step's ids at list index (n - 1) & 1
                const int32_t* __restrict__ src = a.spike_list + (size_t)((n - 1) & 3) * a.N;
                int32_t* __restrict__ dst = a.spike_list + (size_t)((n - 1) & 1) * a.N;
                for (int i = threadIdx.x - U; i < M_last; i += R) dst[i] = __ldcg(src + i);
            }
            if ((int)threadIdx.x == U) {                           // what the other kernels and the host expect to find
                a.ctl->rec_total[n & 1] = rec_prev;
                a.ctl->rec_total[(n - 1) & 1] = rec_prev;
                a.ctl->spikes += spikes;
                a.ctl->spike_cnt[(n - 1) & 3] = M_last;
                a.ctl->spike_cnt[n & 3] = 0;
                a.ctl->step_d = n - 1;
                a.ctl->slot = slot;
                a.ctl->step_u = n;
            }
        }
    }
}

// ------------------------------- stand-alone kernels ---------------------------------
struct WindowShared { unsigned long long off[kMaxWindowSteps + 1]; int W; };

// offsets of the window of step n: steps n-W+1 .. n (W = min(D, n+1)) and the end = start of step n + M
__device__ __forceinline__ void stage_window(const StepArgs& a, long long n, int M, WindowShared& ws) {
    const int D = a.D;
    const int W = (int)(n + 1 < (long long)D ? n + 1 : (long long)D);
    for (int k = threadIdx.x; k <= W; k += blockDim.x) {
        const long long s = n - W + 1 + (k < W ? k : W - 1);
        const unsigned long long v = __ldcg(&a.ctl->win_start[(unsigned long long)s % (unsigned)(D + 1)]);
        ws.off[k] = k < W ? v : v + (unsigned long long)M;
    }
    if (threadIdx.x == 0) ws.W = W;
    __syncthreads();
}
// one thread, after the offsets are staged: publish the start of step n+1 and flag an overflow of the window
__device__ __forceinline__ void window_bookkeeping(const StepArgs& a, long long n, const WindowShared& ws) {
    a.ctl->win_start[(unsigned long long)(n + 1) % (unsigned)(a.D + 1)] = ws.off[ws.W];
    if (ws.off[ws.W] - ws.off[0] > (unsigned long long)a.win_cap) a.ctl->err_window = 1;
}

template <bool kAdex>
__global__ void __launch_bounds__(kUpdateThreads) update_kernel(const NG_GC StepArgs a) {
    __shared__ PopDev sh_pops[kMaxPopsSmem];
    __shared__ StepScalars sc;
    __shared__ unsigned long long win_base;
    if (threadIdx.x == 0) {
        sc.n = __ldcg(&a.ctl->step_u);
        sc.slot = __ldcg(&a.ctl->slot);
        sc.rec_base = __ldcg(&a.ctl->rec_total[sc.n & 1]);
        win_base = a.win_id ? __ldcg(&a.ctl->win_start[(unsigned long long)sc.n % (unsigned)(a.D + 1)]) : 0ULL;
        if (blockIdx.x == 0) {
            a.ctl->step_d = sc.n; a.ctl->slot_d = sc.slot;
            // event-queue backend: the queue of arrival step n was drained by the delivery of step n-1 and is appended
            // to again (as arrival step n + D) by the delivery of this step
            if (a.q_tail) a.q_tail[(size_t)(sc.n % a.D) * kQTailStride] = 0ULL;
        }
    }
    const PopDev* P = stage_pops(a, sh_pops);              // contains the __syncthreads that publishes sc
    if (a.n_pops > kMaxPopsSmem) __syncthreads();
    update_phase<kAdex>(a, P, sc.n, sc.slot, sc.rec_base, (long long)blockIdx.x * blockDim.x + threadIdx.x, (long long)gridDim.x * blockDim.x,
                 win_base);
}

// kKernel 1: row-chunk walk, 2: delay-major segment walk, 4: spike-buffer backend (segment walk over the spike window)
template <int kKernel>
__global__ void __launch_bounds__(kDeliverThreads, 3) deliver_kernel(const NG_GC StepArgs a) {
    __shared__ DeliverShared sh;
    __shared__ StepScalars sc;
    __shared__ WindowShared ws;
    if (threadIdx.x == 0) {
        sc.n = __ldcg(&a.ctl->step_d);
        sc.slot = __ldcg(&a.ctl->slot_d);
        if (kKernel != 1) sc.M = __ldcg(&a.ctl->spike_cnt[sc.n & 3]);
    }
    __syncthreads();
    const long long gtid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long gthreads = (long long)gridDim.x * blockDim.x;
    int M;
    if (kKernel == 1) M = deliver_rows_phase(a, sc.n, sc.slot, sh);
    else if (kKernel == 2) { M = sc.M; deliver_groups_phase<false>(a, sc.n, sc.slot, M, gtid >> 5, gthreads >> 5, threadIdx.x & 31); }
    else {
        M = sc.M;
        stage_window(a, sc.n, M, ws);
        deliver_groups_phase<true>(a, sc.n, sc.slot, M, gtid >> 5, gthreads >> 5, threadIdx.x & 31, ws.off, ws.W);
        if (gtid == 0) window_bookkeeping(a, sc.n, ws);
    }
    if (gtid == 0) bookkeeping_scalar(a, sc.n, sc.slot, M, __ldcg(&a.ctl->rec_total[sc.n & 1]));
}

// ---------------------------------------------------------------------------------------
// Target-sharded multi-GPU ("a spike buffer, similar to the local one, is
// created in the remote host"): rank r owns the neurons [id_first, id_first + N) — their state, their input planes and
// every connection onto them, stored source-major over ALL sources.  One exchange per time step: after update(n) every
// rank stores the ids of ITS spikes straight into the receive buffer of every peer (peer-mapped device memory over
// NVLink: plain stores, then a system-scope release of a step-stamped flag) and then appends what the peers stored in its
// own buffer to its spike array (acquire-poll on the flags); delivery is local.  No collective library call, no host
// round trip.  Receive buffer of a rank: header { int64 flag[2][16]; int32 cnt[2][16]; } padded to 512 B, then
// int32 ids[2][world][cap], indexed by step parity and SOURCE rank.  Two parities suffice: rank s can publish step n+2
// only after it gathered step n+1, i.e. after this rank published n+1, i.e. after this rank gathered step n.
// ---------------------------------------------------------------------------------------
constexpr int kMaxShards = 16;
constexpr int kXchgHeaderBytes = 512;
__device__ __forceinline__ long long* xchg_flag(unsigned char* base, int parity, int src) { return reinterpret_cast<long long*>(base) + parity * kMaxShards + src; }
__device__ __forceinline__ int32_t* xchg_cnt(unsigned char* base, int parity, int src) { return reinterpret_cast<int32_t*>(base + 256) + parity * kMaxShards + src; }
__device__ __forceinline__ int32_t* xchg_ids(unsigned char* base, int parity, int src, int world, int cap) {
    return reinterpret_cast<int32_t*>(base + kXchgHeaderBytes) + ((size_t)parity * world + src) * (size_t)cap;
}

// one CTA per peer: this rank's spikes of step n -> the peer's receive buffer
__global__ void __launch_bounds__(256) xchg_publish_kernel(const StepArgs a) {
    const int q = blockIdx.x;
    if (q == a.xchg_rank) return;
    __shared__ long long n_s; __shared__ int M_s;
    if (threadIdx.x == 0) { n_s = __ldcg(&a.ctl->step_d); M_s = __ldcg(&a.ctl->spike_cnt[n_s & 3]); }
    __syncthreads();
    const long long n = n_s; const int M = M_s, par = (int)(n & 1);
    const int32_t* __restrict__ list = a.spike_list + (size_t)par * a.NS;
    int32_t* dst = xchg_ids(a.xchg[q], par, a.xchg_rank, a.xchg_world, a.xchg_cap);
    for (int i = threadIdx.x; i < M; i += blockDim.x) dst[i] = __ldcg(list + i);
    __threadfence_system();
    __syncthreads();
    if (threadIdx.x == 0) {
        *xchg_cnt(a.xchg[q], par, a.xchg_rank) = M;
        const long long stamp = n + 1;
        asm volatile("st.release.sys.global.s64 [%0], %1;" ::"l"(xchg_flag(a.xchg[q], par, a.xchg_rank)), "l"(stamp) : "memory");
    }
}

// one CTA per peer: the peer's spikes of step n, from this rank's own receive buffer, appended to the spike array
__global__ void __launch_bounds__(256) xchg_gather_kernel(const StepArgs a) {
    const int src = blockIdx.x;
    if (src == a.xchg_rank) return;
    __shared__ long long n_s; __shared__ int M_s, base_s; __shared__ unsigned long long win_s, rec_s;
    unsigned char* own = a.xchg[a.xchg_rank];
    if (threadIdx.x == 0) {
        const long long n = __ldcg(&a.ctl->step_d);
        const int par = (int)(n & 1);
        long long v = 0;
        const long long t0 = clock64();
        do {                                                   // bounded: a lost peer must not hang the GPU
            asm volatile("ld.acquire.sys.global.s64 %0, [%1];" : "=l"(v) : "l"(xchg_flag(own, par, src)) : "memory");
        } while (v != n + 1 && clock64() - t0 < 20000000000LL);
        int M = 0;
        if (v == n + 1) M = *reinterpret_cast<volatile int32_t*>(xchg_cnt(own, par, src)); else a.ctl->err_xchg = 1;
        n_s = n; M_s = M;
        base_s = M > 0 ? atomicAdd(&a.ctl->spike_cnt[n & 3], M) : 0;
        win_s = a.win_id ? __ldcg(&a.ctl->win_start[(unsigned long long)n % (unsigned)(a.D + 1)]) : 0ULL;
        rec_s = __ldcg(&a.ctl->rec_total[n & 1]);
    }
    __syncthreads();
    const long long n = n_s; const int M = M_s, base = base_s, par = (int)(n & 1);
    const int32_t* ids = xchg_ids(own, par, src, a.xchg_world, a.xchg_cap);
    for (int i = threadIdx.x; i < M; i += blockDim.x) {
        const int32_t id = __ldcv(ids + i);
        const size_t k = (size_t)par * a.NS + base + i;
        a.spike_list[k] = id;
        st_row_info(a.spike_row + k, ld_row_info(a.row_info + id));
        if (a.win_id) a.win_id[(win_s + (unsigned long long)(base + i)) % (unsigned long long)a.win_cap] = id;
        // the spike record of every rank holds the spikes of the whole network (the step bookkeeping counts all of them)
        const unsigned long long pos = rec_s + (unsigned long long)(base + i);
        if (pos < (unsigned long long)a.rec_cap) { a.rec_id[pos] = id; a.rec_step[pos] = (int32_t)n; }
    }
}

// Delivery kernel 5 as a stand-alone launch (one per time step, after update_kernel).
__global__ void __launch_bounds__(kQThreads, 1024 / kQThreads) queue_deliver_kernel(const NG_GC StepArgs a) {
    __shared__ QueueShared sh;
    __shared__ StepScalars sc;
    if (threadIdx.x == 0) {
        sc.n = __ldcg(&a.ctl->step_d);
        sc.slot = __ldcg(&a.ctl->slot_d);
        sc.M = __ldcg(&a.ctl->spike_cnt[sc.n & 3]);
        sh.nmodD = (int)(sc.n % a.D);
    }
    __syncthreads();
    float* __restrict__ plane1 = a.ring + (size_t)(sc.slot == 0 ? 1 : 0) * a.NR;       // two planes: this step's and the next step's input
#ifdef NG_Q_SKIP_DRAIN
    queue_append_phase(a, sc.n, sc.M, plane1, sh);
#else
    if (blockIdx.x & 1) { queue_append_phase(a, sc.n, sc.M, plane1, sh); queue_drain_phase(a, plane1, sh); }
    else { queue_drain_phase(a, plane1, sh); queue_append_phase(a, sc.n, sc.M, plane1, sh); }
#endif
    if (blockIdx.x == 0 && threadIdx.x == 0) bookkeeping_scalar(a, sc.n, sc.slot, sc.M, __ldcg(&a.ctl->rec_total[sc.n & 1]));
}

// Event-queue backend, read-back only (NG_FIELD_RING): add the queued events of the pending arrival steps n+1 .. n+D-1 to
// a [D][NR] ring image (the plane of step n itself is copied by the host).
__global__ void materialize_queues_kernel(const StepArgs a, long long n, float* __restrict__ out) {
    const int D = a.D;
    const long long gtid = (long long)blockIdx.x * blockDim.x + threadIdx.x, gthreads = (long long)gridDim.x * blockDim.x;
    for (int k = 1; k < D; ++k) {
        const int qs = (int)((n + k) % D);
        const unsigned long long T0 = a.q_tail[(size_t)qs * kQTailStride];
        const long long T = (long long)(T0 < (unsigned long long)a.q_cap ? T0 : (unsigned long long)a.q_cap);
        for (long long i = gtid; i < T; i += gthreads) {
            const int2 e = a.q_ev[(size_t)qs * (size_t)a.q_cap + i];
            atomicAdd(out + (size_t)qs * a.NR + e.x, __int_as_float(e.y));
        }
    }
}

// One persistent cooperative kernel for n_steps steps: the two phases separated by grid-wide barriers (grid_barrier)
// instead of kernel boundaries (the per-step work of the microcircuit is a few microseconds).
// One CTA per SM keeps the number of barrier arrivals (atomics on one address) at the SM count.
template <int kKernel>
__global__ void __launch_bounds__(kPersistentThreads, 1) persistent_kernel(const NG_GC StepArgs a, long long n_steps) {
    const long long gtid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long gthreads = (long long)gridDim.x * blockDim.x;
    __shared__ PopDev sh_pops[kMaxPopsSmem];
    __shared__ DeliverShared sh;
    __shared__ StepScalars sc;
    __shared__ WindowShared ws;
    __shared__ unsigned long long win_base_sh;
    if (threadIdx.x == 0) {
        sc.n = __ldcg(&a.ctl->step_u);
        sc.slot = __ldcg(&a.ctl->slot);
        sc.rec_base = __ldcg(&a.ctl->rec_total[sc.n & 1]);
        win_base_sh = a.win_id ? __ldcg(&a.ctl->win_start[(unsigned long long)sc.n % (unsigned)(a.D + 1)]) : 0ULL;
    }
    const PopDev* P = stage_pops(a, sh_pops);
    if (a.n_pops > kMaxPopsSmem) __syncthreads();
    long long n = sc.n;
    int slot = sc.slot;
    unsigned long long rec_base = sc.rec_base, spikes = 0, epoch = 0, win_base = win_base_sh;
    for (long long s = 0; s < n_steps; ++s, ++n) {
        // the counter of step n+1 was last read (as step n-3's) before the barriers of step n-1
        if (gtid == 0) a.ctl->spike_cnt[(n + 1) & 3] = 0;
        trace_stamp(a, n, 0);
        update_phase<false>(a, P, n, slot, rec_base, gtid, gthreads, win_base);      // two-phase persistent kernels: LIF only
        trace_stamp(a, n, 1);
        grid_barrier(a.ctl, epoch);
        trace_stamp(a, n, 2);
        int M;
        if (kKernel == 1) M = deliver_rows_phase(a, n, slot, sh);
        else {
            if (threadIdx.x == 0) sc.M = __ldcg(&a.ctl->spike_cnt[n & 3]);
            __syncthreads();
            M = sc.M;
            if (kKernel == 2) deliver_groups_phase<false>(a, n, slot, M, gtid >> 5, gthreads >> 5, threadIdx.x & 31);
            else {
                stage_window(a, n, M, ws);
                deliver_groups_phase<true>(a, n, slot, M, gtid >> 5, gthreads >> 5, threadIdx.x & 31, ws.off, ws.W);
                if (gtid == 0) window_bookkeeping(a, n, ws);
            }
            __syncthreads();                               // sc.M and the window offsets are rewritten next step
        }
        rec_base += (unsigned long long)M; spikes += (unsigned long long)M; win_base += (unsigned long long)M;
        trace_stamp(a, n, 3);
        grid_barrier(a.ctl, epoch);
        trace_stamp(a, n, 5);
        slot = slot + 1 == a.Dr ? 0 : slot + 1;
    }
    if (gtid == 0) {                                       // nobody reads these words any more in this launch
        a.ctl->rec_total[n & 1] = rec_base;
        a.ctl->spikes += spikes;
        a.ctl->step_d = n - 1;
        a.ctl->slot = slot;
        a.ctl->step_u = n;
    }
}

// Spike-buffer backend, read-back only (NG_FIELD_RING): expand the pending part of the spike window into a [D][N] ring
// image: entry (step s, source j), record (target, w, d) with s + d > n arrives in step s + d (slot (s+d) mod D).
__global__ void materialize_window_kernel(const StepArgs a, long long n, float* __restrict__ out) {
    const int D = a.D;
    const int W = (int)(n < (long long)D ? n : (long long)D);                      // steps n-W .. n-1 are buffered
    const int lane = threadIdx.x & 31;
    const long long gwarp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, gwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (int k = 0; k < W; ++k) {
        const long long s = n - W + k;
        const unsigned long long b0 = a.ctl->win_start[(unsigned long long)s % (unsigned)(D + 1)];
        const unsigned long long b1 = a.ctl->win_start[(unsigned long long)(s + 1) % (unsigned)(D + 1)];
        for (unsigned long long pos = b0 + (unsigned long long)gwarp; pos < b1; pos += (unsigned long long)gwarps) {
            const int j = a.win_id[pos % (unsigned long long)a.win_cap];
            const long long r0 = a.row_off[j];
            const int deg = (int)a.grp_rel[(size_t)j * (D + 1) + D];
            for (int q = lane; q < deg; q += 32) {
                const int d = a.dly[r0 + q];
                if (s + d >= n + 1) atomicAdd(out + (size_t)((s + d) % D) * a.NR + a.tgt[r0 + q], a.w[r0 + q]);
            }
        }
    }
}

// Statistics read-out.  rate = spikes / T; CV ISI = std / mean of the inter-spike intervals (population standard deviation,
// PAPER.md:185), NaN with fewer than two intervals.
__global__ void stat_rate_cv_kernel(int N, const int32_t* __restrict__ cnt, const double* __restrict__ sum,
                                    const double* __restrict__ sumsq, double T_s, float* __restrict__ rate, float* __restrict__ cv) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int c = cnt[i];
    rate[i] = (float)((double)c / T_s);
    const int m = c - 1;
    float out = __int_as_float(0x7fc00000);
    if (m >= 2) {
        const double mean = sum[i] / m, var = sumsq[i] / m - mean * mean;
        out = (float)(sqrt(var > 0.0 ? var : 0.0) / mean);
    }
    cv[i] = out;
}
// Pearson correlation of the binned trains of one population's sample:
// C[i,j] = <b_i - mu_i, b_j - mu_j> / sqrt(<b_i - mu_i, b_i - mu_i> <b_j - mu_j, b_j - mu_j>).  One warp per pair.
__global__ void stat_corr_kernel(const uint16_t* __restrict__ bins, int ns, int nb, int stride, float* __restrict__ C) {
    const int lane = threadIdx.x & 31;
    const long long gw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long pair = gw; pair < (long long)ns * ns; pair += nw) {
        const int i = (int)(pair / ns), j = (int)(pair % ns);
        const uint16_t* __restrict__ bi = bins + (size_t)i * stride;
        const uint16_t* __restrict__ bj = bins + (size_t)j * stride;
        double si = 0, sj = 0, sii = 0, sjj = 0, sij = 0;
        for (int b = lane; b < nb; b += 32) {
            const double x = bi[b], y = bj[b];
            si += x; sj += y; sii += x * x; sjj += y * y; sij += x * y;
        }
        for (int o = 16; o > 0; o >>= 1) {
            si += __shfl_xor_sync(0xffffffffu, si, o); sj += __shfl_xor_sync(0xffffffffu, sj, o);
            sii += __shfl_xor_sync(0xffffffffu, sii, o); sjj += __shfl_xor_sync(0xffffffffu, sjj, o);
            sij += __shfl_xor_sync(0xffffffffu, sij, o);
        }
        if (lane == 0) {
            const double cov = sij - si * sj / nb, vi = sii - si * si / nb, vj = sjj - sj * sj / nb;
            C[pair] = (vi > 0 && vj > 0) ? (float)(cov / sqrt(vi * vj)) : __int_as_float(0x7fc00000);
        }
    }
}

__global__ void fill_pop_of_kernel(uint8_t* pop_of, float* V, int first, int n, uint8_t pop, float E_L) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { pop_of[first + i] = pop; V[first + i] = E_L; }
}

}  // namespace ng

// ---------------------------------------------------------------------------------------
// Ceiling probes (ng_probe): what the memory system of this GPU sustains for the access shapes of a3, measured
// with the same instructions the delivery kernels use.  Not on the hot path; bench.py --probe reports them.
// ---------------------------------------------------------------------------------------
namespace ng {
__device__ __forceinline__ uint32_t probe_hash(uint32_t x) {
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16; return x;
}
// kind 0: coalesced 128-bit read stream over `n4` int4 elements
__global__ void probe_stream_kernel(const int4* __restrict__ a, long long n4, int* sink) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    int acc = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
        const int4 t = ld_stream_s32x4((const int32_t*)(a + i));
        acc += t.x ^ t.y ^ t.z ^ t.w;
    }
    if (acc == 0x12345) *sink = acc;
}
// kind 1: `per_thread` red.global.add.f32 per thread to uniformly random cells of ring[0..M)
__global__ void probe_red_kernel(float* ring, uint32_t M, int per_thread) {
    uint32_t s = probe_hash((blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 1u);
    for (int i = 0; i < per_thread; ++i) {
        s = s * 1664525u + 1013904223u;
        red_add_f32(ring + __umulhi(probe_hash(s), M), 1.0f);
    }
}
// kind 2: streamed records (int4 targets + float4 weights, 8 B per event) with one red per event
__global__ void probe_deliver_kernel(const int4* __restrict__ tgt, const float4* __restrict__ w, float* ring, long long n4) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
        const int4 t = ld_stream_s32x4((const int32_t*)(tgt + i));
        const float4 ww = ld_stream_f32x4((const float*)(w + i));
        red_add_f32(ring + t.x, ww.x); red_add_f32(ring + t.y, ww.y);
        red_add_f32(ring + t.z, ww.z); red_add_f32(ring + t.w, ww.w);
    }
}
__global__ void probe_fill_targets_kernel(int32_t* t, long long n, uint32_t M) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        t[i] = (int32_t)__umulhi(probe_hash((uint32_t)i * 2654435761u + (uint32_t)(i >> 32) + 7u), M);
}
}  // namespace ng
