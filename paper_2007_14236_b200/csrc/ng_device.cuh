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

namespace ng {
namespace cg = cooperative_groups;

// counter word 3 of the Philox stream (C1)
enum : uint32_t { kTagConn = 1, kTagPoisson = 2, kTagInject = 3 };
enum : int32_t { kRuleIndegree = 0, kRuleOutdegree = 1 };
enum : int32_t { kDistConst = 0, kDistNormalClipped = 1, kDistUniformInt = 2 };

constexpr int kMaxPoissonTable = 64;
constexpr int kUpdateThreads = 256;
constexpr int kDeliverThreads = 256;
constexpr int kChunkRecords = 128;   // records one warp consumes per iteration of the row walk: 32 lanes x 4

struct DistDev { int32_t kind; int32_t pad; double a, b, lo, hi; };

struct CallDev {               // one ng_connect_* call
    int32_t rule, src_first, src_n, tgt_first, tgt_n, K;
    int32_t call_index, pad;
    DistDev w, d;
};

struct PopDev {                // per-population constants of the update (fp32 copies of fp64 host values)
    float P11, P22, P21, P20Ie;            // exact-integration propagators; P20Ie = P20 * I_e
    float E_L, V_th, V_reset, w_ext;
    int32_t refr_steps, n_T;
    uint32_t T[kMaxPoissonTable];          // integer Poisson CDF table (C7)
};

struct Ctl {                   // device-resident control block; see ng.cu for the update/deliver handshake
    long long step_u;                      // written by deliver, read by update: index of the next step
    long long step_d;                      // written by update, read by deliver: index of the step being delivered
    int32_t spike_cnt[4];                  // length of the spike array of step n, indexed n & 3 (the list itself by n & 1)
    unsigned long long rec_total[2];       // spikes recorded before step of this parity
    unsigned long long spikes, events;
    int32_t err_delay;                     // builder: a drawn delay fell outside [1, D]
    int32_t max_row_records;               // builder: longest padded row
    unsigned long long n_padded;           // builder: total records stored
    unsigned int ticket;                   // fused step kernel: CTAs that finished the current step
    unsigned int pad0;
    unsigned long long bar;                // persistent fused kernel: arrivals at the grid barrier
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
                   uint32_t* __restrict__ cnt, Ctl* __restrict__ ctl) {
    const CallDev c = calls[call_idx];
    const int32_t e_first = c.rule == kRuleIndegree ? c.tgt_first : c.src_first;
    const int32_t e_n = c.rule == kRuleIndegree ? c.tgt_n : c.src_n;
    const long long total = (long long)e_n * c.K;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += stride) {
        const int32_t e = e_first + (int32_t)(idx / c.K);
        const int32_t k = (int32_t)(idx % c.K);
        const Draw dr = draw_connection<false>(c, seed_lo, seed_hi, e, k);
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
    if (j < N) {
        for (int d = 0; d < D; ++d) len += (int)cnt[(size_t)j * D + d];
        len = (len + 3) & ~3;
        row_len[j] = len;
    }
    // block max -> one atomic per block
    __shared__ int smax;
    if (threadIdx.x == 0) smax = 0;
    __syncthreads();
    atomicMax(&smax, len);
    __syncthreads();
    if (threadIdx.x == 0) atomicMax(&ctl->max_row_records, smax);
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

__global__ void __launch_bounds__(256)
build_fill_kernel(const CallDev* __restrict__ calls, int call_idx, uint32_t seed_lo, uint32_t seed_hi, int D,
                  uint32_t* __restrict__ cursor, const long long* __restrict__ row_off,
                  const uint32_t* __restrict__ grp_rel, int32_t* __restrict__ tgt, float* __restrict__ w,
                  uint8_t* __restrict__ dly) {
    const CallDev c = calls[call_idx];
    const int32_t e_first = c.rule == kRuleIndegree ? c.tgt_first : c.src_first;
    const int32_t e_n = c.rule == kRuleIndegree ? c.tgt_n : c.src_n;
    const long long total = (long long)e_n * c.K;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += stride) {
        const int32_t e = e_first + (int32_t)(idx / c.K);
        const int32_t k = (int32_t)(idx % c.K);
        const Draw dr = draw_connection<true>(c, seed_lo, seed_hi, e, k);
        if (dr.delay < 1 || dr.delay > D) continue;
        const uint32_t p = atomicAdd(&cursor[(size_t)dr.src * D + (dr.delay - 1)], 1u);
        const long long pos = row_off[dr.src] + grp_rel[(size_t)dr.src * (D + 1) + (dr.delay - 1)] + p;
        tgt[pos] = dr.tgt;
        w[pos] = dr.w;
        dly[pos] = (uint8_t)dr.delay;
    }
}

// Order the records of every (source, delay) group by (target, weight bits): the fill order above depends on
// atomic arrival order; after this pass the structure is a deterministic function of the seed.
// One warp per group; groups are short (1..~1e3 records), so an in-place odd-even transposition over
// lane-strided elements is enough.  Groups longer than kSortMax records are left as filled.
constexpr int kSortMax = 768;    // 8 warps x 768 x 8 B = 48 KB of static shared memory
__global__ void __launch_bounds__(256)
build_sort_groups_kernel(int N, int D, const long long* __restrict__ row_off, const uint32_t* __restrict__ grp_rel,
                         int32_t* __restrict__ tgt, float* __restrict__ w) {
    __shared__ unsigned long long keys[8][kSortMax];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const long long n_groups = (long long)N * D;
    const long long warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long g = (((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5); g < n_groups; g += warps) {
        const int j = (int)(g / D), d = (int)(g % D);
        const uint32_t a = grp_rel[(size_t)j * (D + 1) + d], b = grp_rel[(size_t)j * (D + 1) + d + 1];
        const int len = (int)(b - a);
        if (len < 2 || len > kSortMax) continue;
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

// ---------------------------------------------------------------------------------------
// Warp-aggregated append to the spike array (Fig. 1b: "the spike is sent to the spike
// array"; its maximum size is the number of nodes).  One atomicAdd per warp that holds a spike.
// Every lane of the warp must call this.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void append_spike(bool spk, int32_t id, int32_t* __restrict__ list, int32_t* cnt) {
    const unsigned m = __ballot_sync(0xffffffffu, spk);
    if (m == 0) return;
    const int lane = threadIdx.x & 31;
    const int leader = __ffs(m) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(cnt, __popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (spk) list[base + __popc(m & ((1u << lane) - 1u))] = id;
}

struct StepArgs {
    int32_t N, D;                // D = ring_slots of the C-ABI = largest legal delay
    int32_t Dr, n_pops;          // Dr = D + 1 planes are stored (see update_phase); number of populations
    uint32_t seed_lo, seed_hi;
    // neuron state (SoA) and parameters
    float* V; float* I; int32_t* refr; const uint8_t* pop_of; const PopDev* pops;
    float* ring;                 // [Dr][N] slot-major
    float* last_input;           // [N] or nullptr (NG_DEBUG_INPUT)
    // spike array, double-buffered by step parity, and the spike record
    int32_t* spike_list;         // [2][N]
    int32_t* rec_step; int32_t* rec_id; long long rec_cap;   // rec_cap = 0: recording off
    // connection structure
    const long long* row_off; const uint32_t* grp_rel;
    const int32_t* tgt; const float* w; const uint8_t* dly;
    Ctl* ctl;
    int32_t bypass; uint32_t inject_thr;
    int32_t max_row_chunks;      // ceil(longest padded row / kChunkRecords)
};

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
__device__ __forceinline__ bool neuron_step(const StepArgs& a, const PopDev* __restrict__ P, long long n, int i,
                                            float* __restrict__ plane) {
    // all independent loads first: one memory round trip instead of a chain
    const float in = __ldcg(plane + i);          // written by red.global from other SMs: read at L2
    if (a.bypass) {                                          // DESIGN.md C8: delivery-only mode
        plane[i] = 0.f;
        if (a.last_input) a.last_input[i] = in;
        const uint4 x = philox4x32_10(a.seed_lo, a.seed_hi, (uint32_t)i, (uint32_t)n, (uint32_t)(n >> 32), kTagInject);
        return x.x < a.inject_thr;
    }
    float V = a.V[i], I = a.I[i];
    int r = a.refr[i];
    const int pi = a.pop_of[i];
    plane[i] = 0.f;
    if (a.last_input) a.last_input[i] = in;
    const PopDev* __restrict__ p = P + pi;
    int k = 0;
    const int nT = p->n_T;
    if (nT > 0) {
        const uint4 x = philox4x32_10(a.seed_lo, a.seed_hi, (uint32_t)i, (uint32_t)n, (uint32_t)(n >> 32), kTagPoisson);
        while (k < nT && x.x >= p->T[k]) ++k;                // T is non-decreasing: k = #{m : x0 >= T[m]}
    }
    const float E_L = p->E_L;
    bool spk = false;
    if (r == 0) V = E_L + fmaf(p->P22, V - E_L, fmaf(p->P21, I, p->P20Ie));
    else r -= 1;
    I = fmaf(p->P11, I, in) + p->w_ext * (float)k;
    if (V >= p->V_th) { spk = true; V = p->V_reset; r = p->refr_steps; }
    a.V[i] = V; a.I[i] = I; a.refr[i] = r;
    return spk;
}

__device__ __forceinline__ void update_phase(const StepArgs& a, const PopDev* __restrict__ P, long long n, long long gtid,
                                             long long gthreads) {
    const int N = a.N;
    const int slot = (int)(n % a.Dr);
    float* __restrict__ plane = a.ring + (size_t)slot * N;
    int32_t* __restrict__ list = a.spike_list + (size_t)(n & 1) * N;
    int32_t* cnt = &a.ctl->spike_cnt[n & 3];
    const long long n_round = ((long long)N + 31) & ~31LL;      // keep warps whole for the ballot
    for (long long ii = gtid; ii < n_round; ii += gthreads) {
        const int i = (int)ii;
        const bool spk = i < N && neuron_step(a, P, n, i, plane);
        append_spike(spk, i, list, cnt);
    }
    if (gtid == 0) a.ctl->step_d = n;
}

__device__ __forceinline__ void red_add_f32(float* addr, float v) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ int4 ld_stream_s32x4(const int32_t* p) {
    int4 r;
    asm("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ float4 ld_stream_f32x4(const float* p) {
    float4 r;
    asm("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ uint32_t ld_stream_u32(const void* p) {
    uint32_t r;
    asm("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(r) : "l"(p));
    return r;
}

// Step bookkeeping shared by both delivery kernels (a4): one thread publishes the next step index, clears the
// other parity's spike counter and advances the record cursor; all threads copy the spike array into the
// spike record (a2, "all spike times of all neurons recorded").
__device__ __forceinline__ void bookkeeping_phase(const StepArgs& a, long long n, int M, long long gtid, long long gthreads) {
    const unsigned long long rec_base = __ldcg(&a.ctl->rec_total[n & 1]);
    if (a.rec_cap > 0) {
        const int32_t* __restrict__ list = a.spike_list + (size_t)(n & 1) * a.N;
        for (long long i = gtid; i < M; i += gthreads) {
            const unsigned long long pos = rec_base + (unsigned long long)i;
            if (pos < (unsigned long long)a.rec_cap) { a.rec_id[pos] = __ldcg(list + i); a.rec_step[pos] = (int32_t)n; }
        }
    }
    if (gtid == 0) {
        a.ctl->rec_total[(n + 1) & 1] = rec_base + (unsigned long long)M;
        a.ctl->spike_cnt[(n + 1) & 3] = 0;
        a.ctl->spikes += (unsigned long long)M;
        a.ctl->step_u = n + 1;
    }
}

// ---------------------------------------------------------------------------------------
// a3. Spike delivery, kernel 1: row-chunk walk.
//   work item = (spike index i, chunk c of kChunkRecords records of row(spike i)), chunk fastest, one warp per
//   item; lane l reads records [4l, 4l+4) of the chunk with one 128-bit load of targets, one of weights and one
//   32-bit load of delays, then issues up to four red.global.add.f32 into ring[(n + d) mod D][target].
//   Rows are delay-grouped, so consecutive records mostly hit the same ring plane.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void deliver_rows_phase(const StepArgs& a, long long n, int M, long long gwarp, long long gwarps,
                                                   int lane) {
    const int N = a.N, D = a.D, Dr = a.Dr;
    const int nmod = (int)(n % Dr);
    const int32_t* __restrict__ list = a.spike_list + (size_t)(n & 1) * N;
    const int chunks = a.max_row_chunks;
    const long long items = (long long)M * chunks;
    unsigned long long ev = 0;
    for (long long it = gwarp; it < items; it += gwarps) {
        const int si = (int)(it / chunks), c = (int)(it % chunks);
        const int j = __ldcg(list + si);
        const long long r0 = a.row_off[j], r1 = a.row_off[j + 1];
        if (c == 0 && lane == 0) ev += a.grp_rel[(size_t)j * (D + 1) + D];
        const long long p = r0 + (long long)c * kChunkRecords + lane * 4;
        if (p < r1) {
            const int4 t = ld_stream_s32x4(a.tgt + p);
            const float4 ww = ld_stream_f32x4(a.w + p);
            const uint32_t dd = ld_stream_u32(a.dly + p);
            int s;
            if (t.x >= 0) { s = nmod + (int)(dd & 0xff); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * N + t.x, ww.x); }
            if (t.y >= 0) { s = nmod + (int)((dd >> 8) & 0xff); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * N + t.y, ww.y); }
            if (t.z >= 0) { s = nmod + (int)((dd >> 16) & 0xff); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * N + t.z, ww.z); }
            if (t.w >= 0) { s = nmod + (int)(dd >> 24); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * N + t.w, ww.w); }
        }
    }
    if (ev) atomicAdd(&a.ctl->events, ev);
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
    float* __restrict__ plane = a.ring + (size_t)r.slot * a.N;
    if (r.q >= r.rel_lo && r.q < r.len) red_add_f32(plane + t.x, ww.x);
    if (r.q + 1 >= r.rel_lo && r.q + 1 < r.len) red_add_f32(plane + t.y, ww.y);
    if (r.q + 2 >= r.rel_lo && r.q + 2 < r.len) red_add_f32(plane + t.z, ww.z);
    if (r.q + 3 >= r.rel_lo && r.q + 3 < r.len) red_add_f32(plane + t.w, ww.w);
}

__device__ __forceinline__ void deliver_groups_phase(const StepArgs& a, long long n, int M, long long gwarp, long long gwarps,
                                                     int lane) {
    const int N = a.N, D = a.D, Dr = a.Dr;
    const int nmod = (int)(n % Dr);
    const int32_t* __restrict__ list = a.spike_list + (size_t)(n & 1) * N;
    const long long items = (long long)M * D;
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
        if (small) { d = (int)((uint32_t)it / (uint32_t)M); si = (int)((uint32_t)it - (uint32_t)d * (uint32_t)M); }
        else { d = (int)(it / M); si = (int)(it - (long long)d * M); }
        return true;
    };
    auto load_j = [&](long long b) -> int {
        int d, si;
        return item_of(b, d, si) ? __ldcg(list + si) : -1;
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
            if (d == 0) ev += g[D];
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
            slot = nmod + d_cur + 1; if (slot >= Dr) slot -= Dr;
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

// ---------------------------------------------------------------------------------------
// a1 + a2 + a3 fused: kernel 3, one kernel per time step (the latency regime: tens of spikes per step).
//   Every thread updates one neuron; the CTA gathers its own spikes in shared memory (id, row start, padded row
//   length — the row bounds are fetched by the thread that spiked, so they are in flight while the rest of the CTA
//   finishes its update), appends them to the global spike array / spike record with ONE atomic per CTA, and then
//   walks the rows of its own spikes: 128-bit loads of targets and weights, 32-bit loads of delays, two vectors
//   per thread in flight, red.global.add.f32 into ring[(n + d) mod Dr][target].
//   No grid-wide dependency exists inside the step (the consumed plane n mod Dr is never a delivery target, see
//   neuron_step), so a step costs one launch — or one grid barrier in the persistent variant — instead of two.
// ---------------------------------------------------------------------------------------
constexpr int kFusedThreads = 256;
struct FusedShared {
    PopDev pops[kMaxPopsSmem];
    long long r0[kFusedThreads];
    int32_t len[kFusedThreads];
    int32_t id[kFusedThreads];
    int32_t cnt, gbase;
};

__device__ __forceinline__ void red_rec4(const StepArgs& a, int nmod, const int4& t, const float4& ww, uint32_t dd) {
    const int N = a.N, Dr = a.Dr;
    int s;
    if (t.x >= 0) { s = nmod + (int)(dd & 0xff); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * N + t.x, ww.x); }
    if (t.y >= 0) { s = nmod + (int)((dd >> 8) & 0xff); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * N + t.y, ww.y); }
    if (t.z >= 0) { s = nmod + (int)((dd >> 16) & 0xff); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * N + t.z, ww.z); }
    if (t.w >= 0) { s = nmod + (int)(dd >> 24); if (s >= Dr) s -= Dr; red_add_f32(a.ring + (size_t)s * N + t.w, ww.w); }
}

__device__ __forceinline__ void fused_phase(const StepArgs& a, const PopDev* __restrict__ P, long long n,
                                            unsigned long long rec_base, FusedShared& sh) {
    const int N = a.N, D = a.D;
    const int nmod = (int)(n % a.Dr);
    float* __restrict__ plane = a.ring + (size_t)nmod * N;
    int32_t* __restrict__ list = a.spike_list + (size_t)(n & 1) * N;
    const int lane = threadIdx.x & 31;
    unsigned long long ev = 0;
    for (long long base = (long long)blockIdx.x * kFusedThreads; base < N; base += (long long)gridDim.x * kFusedThreads) {
        __syncthreads();                                   // previous round's readers of sh are done
        if (threadIdx.x == 0) sh.cnt = 0;
        __syncthreads();
        const long long ii = base + threadIdx.x;
        const int i = (int)ii;
        const bool spk = ii < N && neuron_step(a, P, n, i, plane);
        const unsigned m = __ballot_sync(0xffffffffu, spk);
        if (m) {                                           // warp-aggregated append to the CTA's list
            const int leader = __ffs(m) - 1;
            int b = 0;
            if (lane == leader) b = atomicAdd(&sh.cnt, __popc(m));
            b = __shfl_sync(0xffffffffu, b, leader);
            if (spk) {
                const int k = b + __popc(m & ((1u << lane) - 1u));
                const long long r0 = a.row_off[i], r1 = a.row_off[i + 1];
                sh.id[k] = i; sh.r0[k] = r0; sh.len[k] = (int)(r1 - r0);
                ev += a.grp_rel[(size_t)i * (D + 1) + D];
            }
        }
        __syncthreads();
        const int Ml = sh.cnt;
        if (Ml == 0) continue;                             // uniform over the CTA
        if (threadIdx.x == 0) sh.gbase = atomicAdd(&a.ctl->spike_cnt[n & 3], Ml);
        for (int s = 0; s < Ml; ++s) {                     // a3: walk the rows of this CTA's spikes
            const long long r0 = sh.r0[s];
            const int len = sh.len[s];
            for (int p = threadIdx.x * 4; p < len; p += kFusedThreads * 8) {
                const int q = p + kFusedThreads * 4;
                const int4 t0 = ld_stream_s32x4(a.tgt + r0 + p);
                const float4 w0 = ld_stream_f32x4(a.w + r0 + p);
                const uint32_t d0 = ld_stream_u32(a.dly + r0 + p);
                int4 t1 = make_int4(-1, -1, -1, -1); float4 w1 = make_float4(0.f, 0.f, 0.f, 0.f); uint32_t d1 = 0;
                if (q < len) { t1 = ld_stream_s32x4(a.tgt + r0 + q); w1 = ld_stream_f32x4(a.w + r0 + q); d1 = ld_stream_u32(a.dly + r0 + q); }
                red_rec4(a, nmod, t0, w0, d0);
                red_rec4(a, nmod, t1, w1, d1);
            }
        }
        __syncthreads();                                   // sh.gbase
        const int gb = sh.gbase;
        for (int k = threadIdx.x; k < Ml; k += kFusedThreads) {    // a2: spike array and spike record
            const int id = sh.id[k];
            list[gb + k] = id;
            const unsigned long long pos = rec_base + (unsigned long long)(gb + k);
            if (pos < (unsigned long long)a.rec_cap) { a.rec_id[pos] = id; a.rec_step[pos] = (int32_t)n; }
        }
    }
    if (ev) atomicAdd(&a.ctl->events, ev);
}

// One launch = one time step.  The last CTA to finish publishes the next step index (a4).
__global__ void __launch_bounds__(kFusedThreads) fused_step_kernel(const StepArgs a) {
    __shared__ FusedShared sh;
    const long long n = __ldcg(&a.ctl->step_u);
    const unsigned long long rec_base = __ldcg(&a.ctl->rec_total[n & 1]);
    const PopDev* P = stage_pops(a, sh.pops);
    fused_phase(a, P, n, rec_base, sh);
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned t = atomicAdd(&a.ctl->ticket, 1u);
        if (t == gridDim.x - 1) {
            __threadfence();
            const int M = __ldcg(&a.ctl->spike_cnt[n & 3]);
            a.ctl->rec_total[(n + 1) & 1] = rec_base + (unsigned long long)M;
            a.ctl->spike_cnt[(n + 1) & 3] = 0;
            a.ctl->spikes += (unsigned long long)M;
            a.ctl->ticket = 0;
            a.ctl->step_d = n;
            a.ctl->step_u = n + 1;
        }
    }
}

// Grid barrier of the persistent fused kernel: one atomic arrival per CTA on a counter that only grows, then a
// poll.  The kernel is launched cooperatively (all CTAs co-resident); the host clears ctl->bar before the launch.
__device__ __forceinline__ void grid_barrier(Ctl* ctl, unsigned long long& epoch) {
    __syncthreads();
    if (threadIdx.x == 0) {
        epoch += gridDim.x;
        __threadfence();
        atomicAdd(&ctl->bar, 1ULL);
        unsigned long long v;
        do {
            asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(&ctl->bar) : "memory");
        } while (v < epoch);
        __threadfence();
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kFusedThreads) persistent_fused_kernel(const StepArgs a, long long n_steps) {
    __shared__ FusedShared sh;
    long long n = __ldcg(&a.ctl->step_u);
    unsigned long long rec_base = __ldcg(&a.ctl->rec_total[n & 1]);
    unsigned long long epoch = 0, spikes = 0;
    const PopDev* P = stage_pops(a, sh.pops);
    for (long long s = 0; s < n_steps; ++s, ++n) {
        // the counter of step n+1 was last read (as step n-3's) long before the previous barrier
        if (blockIdx.x == 0 && threadIdx.x == 0) a.ctl->spike_cnt[(n + 1) & 3] = 0;
        fused_phase(a, P, n, rec_base, sh);
        grid_barrier(a.ctl, epoch);
        const unsigned long long M = (unsigned long long)__ldcg(&a.ctl->spike_cnt[n & 3]);
        rec_base += M; spikes += M;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {             // nobody reads these words any more in this launch
        a.ctl->rec_total[n & 1] = rec_base;
        a.ctl->spikes += spikes;
        a.ctl->step_d = n - 1;
        a.ctl->step_u = n;
    }
}

// ------------------------------- stand-alone kernels ---------------------------------
__global__ void __launch_bounds__(kUpdateThreads) update_kernel(const StepArgs a) {
    __shared__ PopDev sh_pops[kMaxPopsSmem];
    const long long n = __ldcg(&a.ctl->step_u);
    const PopDev* P = stage_pops(a, sh_pops);
    update_phase(a, P, n, (long long)blockIdx.x * blockDim.x + threadIdx.x, (long long)gridDim.x * blockDim.x);
}

template <int kKernel>
__global__ void __launch_bounds__(kDeliverThreads) deliver_kernel(const StepArgs a) {
    const long long n = __ldcg(&a.ctl->step_d);
    const int M = __ldcg(&a.ctl->spike_cnt[n & 3]);
    const long long gtid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long gthreads = (long long)gridDim.x * blockDim.x;
    if (kKernel == 1) deliver_rows_phase(a, n, M, gtid >> 5, gthreads >> 5, threadIdx.x & 31);
    else deliver_groups_phase(a, n, M, gtid >> 5, gthreads >> 5, threadIdx.x & 31);
    bookkeeping_phase(a, n, M, gtid, gthreads);
}

// One persistent cooperative kernel for n_steps steps: the two phases separated by grid-wide barriers instead of
// kernel boundaries (the per-step work of the microcircuit is a few microseconds).
template <int kKernel>
__global__ void __launch_bounds__(kUpdateThreads) persistent_kernel(const StepArgs a, long long n_steps) {
    cg::grid_group grid = cg::this_grid();
    const long long gtid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long gthreads = (long long)gridDim.x * blockDim.x;
    __shared__ PopDev sh_pops[kMaxPopsSmem];
    const PopDev* P = stage_pops(a, sh_pops);
    long long n = __ldcg(&a.ctl->step_u);
    grid.sync();                                   // everyone has read step_u before anyone moves it
    for (long long s = 0; s < n_steps; ++s, ++n) {
        update_phase(a, P, n, gtid, gthreads);
        grid.sync();
        const int M = __ldcg(&a.ctl->spike_cnt[n & 3]);
        if (kKernel == 1) deliver_rows_phase(a, n, M, gtid >> 5, gthreads >> 5, threadIdx.x & 31);
        else deliver_groups_phase(a, n, M, gtid >> 5, gthreads >> 5, threadIdx.x & 31);
        bookkeeping_phase(a, n, M, gtid, gthreads);
        grid.sync();
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
