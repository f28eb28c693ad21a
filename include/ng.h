/* =====================================================================================
 * ng.h — C-ABI of libng.so: the per-time-step hot path of a clock-driven spiking-network
 * simulator as arXiv 2007.14236 defines it, hand-written CUDA for sm_100a.
 *
 * What the path computes, per step n (t_n -> t_{n+1}, h = dt):
 *   a1  LIF (iaf_psc_exp) exact-integration update fused with a Poisson background drive
 *       PAPER.md:93-102 Eqs. (1)-(2); "integrated by the exact integration scheme
 *       described in [20] on the time grid"; PAPER.md:187 refractory time; C7, C11
 *   a2  spike collection into the global spike array          PAPER.md:69, Fig. 1(b)
 *   a3  spike delivery: every connection (j -> i, w, d) of a neuron j that spiked in step n
 *       adds w to ring slot (n + d) mod D of target i          PAPER.md:69 (delay-ordered
 *       connection groups; "when the time index t_s matches the connection-group delay")
 *   a0  (setup) fixed-indegree / fixed-outdegree connection rules, built directly
 *       in GPU memory (PAPER.md:292 names this as the fix for the build-time bottleneck)
 *
 * Conventions
 *   - every function returns an int32 status (NG_OK = 0, negatives below); nothing throws or aborts.
 *     ng_last_error() gives a message owned by the handle, valid until the next call on it.
 *   - one handle per host thread; no global state.  All device work is enqueued on the CUDA stream
 *     given to ng_create (NULL = the legacy default stream).
 *   - pointers named *_host must be host memory; pointers named `data`/`out` in ng_set_state,
 *     ng_get_state and ng_copy_* may be host OR device memory (unified addressing decides).
 *     Every buffer passed in is caller-owned; the library never frees caller memory.
 *   - device memory comes from the ng_allocator callbacks (the Python harness backs them with
 *     torch tensors); with a NULL allocator cudaMalloc/cudaFree are used.  Everything is released
 *     by ng_destroy.
 *   - neuron ids are global, contiguous, assigned in ng_create_population order.
 *   - time: a spike reported with step n happened at t = (n+1)*h.  A delay of d steps makes the
 *     synaptic current of the target jump at t = (n+1+d)*h (C10).  1 <= d <= ring_slots.
 * ===================================================================================== */
#ifndef NG_H_
#define NG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ng_sim ng_sim;

/* status codes */
enum {
    NG_OK = 0,
    NG_ERR_INVALID_ARG = -1,
    NG_ERR_STATE = -2,      /* call not legal in this state (e.g. connect after prepare) */
    NG_ERR_OOM = -3,
    NG_ERR_CUDA = -4,
    NG_ERR_OVERFLOW = -5    /* spike record full, or a drawn delay outside [1, ring_slots] */
};

/* ng_config.flags */
enum {
    NG_RECORD_SPIKES = 1u << 0,   /* keep (step, id) of every spike on the device until ng_get_spikes */
    NG_DEBUG_INPUT = 1u << 1      /* keep the ring plane consumed by the last step (field NG_FIELD_LAST_INPUT) */
};

/* state fields for ng_set_state / ng_get_state */
enum {
    NG_FIELD_V = 0,           /* float  [N]   membrane potential, mV                               */
    NG_FIELD_I_SYN = 1,       /* float  [N]   synaptic current, pA                                 */
    NG_FIELD_REFR = 2,        /* int32  [N]   remaining refractory steps                           */
    NG_FIELD_RING = 3,        /* float  [D*N] input ring buffer, slot-major: ring[slot*N + i]      */
    NG_FIELD_STEP = 4,        /* int64  [1]   index n of the next step                             */
    NG_FIELD_LAST_INPUT = 5,  /* float  [P*N] in_i consumed by the last step (needs NG_DEBUG_INPUT; get only) */
    /* AdEx state (only with AdEx populations), float [N] each; V is NG_FIELD_V */
    NG_FIELD_ADEX_W = 6,      /* adaptation current w, pA                                           */
    NG_FIELD_ADEX_G_EX = 7,   /* excitatory conductance g_ex, nS                                    */
    NG_FIELD_ADEX_Y_EX = 8,   /* its alpha-function companion y_ex, nS/ms                           */
    NG_FIELD_ADEX_G_IN = 9,   /* inhibitory conductance g_in, nS                                    */
    NG_FIELD_ADEX_Y_IN = 10,  /* y_in, nS/ms                                                        */
    NG_FIELD_ADEX_H = 11      /* current sub-step size of the adaptive integrator, ms               */
};
/* Receptor ports: P = 1, or 2 as soon as an AdEx population exists (port 0 excitatory — also the LIF input current —,
 * port 1 inhibitory).  NG_FIELD_RING is then [D][P][N], NG_FIELD_LAST_INPUT [P][N], and the stored target of a
 * connection record (ng_copy_records, ng_get_connections) is target id + port * N. */

/* distribution kinds for weights and delays ("fixed values ... or probability distributions") */
enum {
    NG_DIST_CONST = 0,          /* value a                                                          */
    NG_DIST_NORMAL_CLIPPED = 1, /* a + b*z, z ~ N(0,1) (fp64 Box-Muller, C4), clipped to [lo, hi];
                                   as a delay: floor(a + b*z + 0.5) clipped to [lo, hi] (C5)   */
    NG_DIST_UNIFORM_INT = 2     /* integer uniform on [lo, hi] (C5)                       */
};

/* options for ng_set_option */
enum {
    NG_OPT_STEP_MODE = 0,        /* 0 = CUDA graph of NG_OPT_STEPS_PER_GRAPH steps, 1 = plain kernel launches,
                                    2 = one persistent cooperative kernel per ng_simulate call,
                                    3 = auto (default): 2 for delivery kernels 1 and 3, 0 for kernel 2      */
    NG_OPT_STEPS_PER_GRAPH = 1,  /* default 100 */
    NG_OPT_DELIVERY_KERNEL = 2,  /* 0 = auto, 1 = row-chunk walk, 2 = delay-major segment walk,
                                    3 = pipelined step kernel (delay-1 records with the update, the rest
                                        overlapped with the next step: one grid dependency per step),
                                    4 = spike-buffer backend, the paper's own mechanism: no D-plane
                                        ring; the spikes of the last ring_slots steps stay buffered and reach their
                                        delay groups one step at a time.  Must be chosen BEFORE ng_prepare;
                                        NG_FIELD_RING is then read-only (expanded on demand),
                                    5 = per-delay event queues: a spiking row is read once and its records are appended,
                                        binned by delay, to the queue of their arrival step; every step streams ONE
                                        queue into the input plane of the next step.  Two planes like kernel 4, same
                                        rules (before ng_prepare, NG_FIELD_RING read-only).  Memory: ring_slots queues
                                        of NG_OPT_QUEUE_CAPACITY events x 8 B; a full queue drops events and
                                        ng_simulate returns NG_ERR_OVERFLOW,
                                    6 = kernel 3's pipelined step with kernel 4's backend: the delay-1 records go out with
                                        the update, the rest warps walk the spike window (one delay group per buffered
                                        spike and step) into the ONE input plane of the next step.  Persistent cooperative
                                        kernel only (step mode 2), one GPU, not in delivery-only mode; rules of kernel 4  */
    NG_OPT_DELIVER_BLOCKS = 3,   /* grid size of the delivery kernel, 0 = auto                         */
    NG_OPT_PROFILE = 4,          /* 1 = time every kernel with CUDA events (forces plain launches);
                                    results in ng_stats.ms_update / ms_deliver                       */
    NG_OPT_ASYNC = 5,            /* 1 = ng_simulate returns after enqueueing (no stream synchronise)   */
    NG_OPT_SORT_SEGMENTS = 6,    /* 1 = order records inside each (source, delay) group by target id
                                    after the build (default 1; must be set before ng_prepare)        */
    NG_OPT_PREFETCH = 7,         /* 1 = the thread that detects a spike bulk-prefetches the spiking row into
                                    L2 (default 1; ignored by delivery kernel 2)                       */
    NG_OPT_TRACE = 8,            /* 1 = the persistent kernels (step mode 2) stamp %globaltimer at every phase
                                    boundary of every CTA; read with ng_get_trace (after ng_prepare)   */
    NG_OPT_PERSISTENT_THREADS = 9, /* threads per CTA of the persistent kernels: 1024 (default, one CTA per SM) or 512 */
    NG_OPT_QUEUE_CAPACITY = 10   /* delivery kernel 5: events per queue (before ng_prepare).  0 = auto: 1.25 x the expected
                                    events per step (delivery-only mode: inject fraction x connections; else 2 % of
                                    the connections, i.e. a mean rate of 200 Hz at dt = 0.1 ms) + 65536              */
};

typedef struct {
    double dt_ms;                 /* h, PAPER.md:181 uses 0.1 ms                                      */
    int32_t ring_slots;           /* D >= largest delay in steps (C9), 1..255               */
    uint32_t flags;               /* NG_RECORD_SPIKES | NG_DEBUG_INPUT                                */
    uint64_t seed;                /* Philox4x32-10 key (C1)                                 */
    int64_t max_recorded_spikes;  /* capacity of the device spike record (used with NG_RECORD_SPIKES) */
    int32_t device;               /* CUDA device ordinal                                              */
    int32_t reserved;
} ng_config;

typedef struct {
    void* (*alloc)(size_t bytes, void* user);   /* returns device memory, 256-byte aligned, or NULL */
    void (*free)(void* ptr, void* user);
    void* user;
} ng_allocator;

/* iaf_psc_exp parameters, symbols of PAPER.md:93-102.  Units: pF, ms, mV, pA, Hz. */
typedef struct {
    double C_m, tau_m, tau_syn, E_L, V_th, V_reset, t_ref_ms, I_e;
    double poisson_rate_hz;   /* total rate of the background drive per neuron (e.g. 8 Hz * K_ext) */
    double poisson_weight;    /* pA per background event                                           */
} ng_lif_params;

/* AdEx neuron with conductance-based alpha synapses, the model of the paper's balanced network (PAPER.md:110-161,
 * Eqs. (3)-(5), Table II symbols).  Units: pF, nS, mV, ms, pA, Hz; weights of connections onto AdEx neurons are peak
 * conductances in nS.  V_peak, tol and h_min are not in the paper (readings C23, C24). */
typedef struct {
    double C_m, g_L, E_L, V_T, Delta_T, tau_w, a, b, V_reset, V_peak, E_ex, E_in, tau_syn, I_e;
    double poisson_rate_hz;   /* background drive onto the excitatory port                           */
    double poisson_weight;    /* nS per background event                                             */
    double tol[6];            /* absolute tolerances of (V, w, g_ex, y_ex, g_in, y_in) for the step-size control */
    double h_min;             /* smallest sub-step of the adaptive Runge-Kutta integrator, ms        */
} ng_adex_params;

typedef struct {
    int32_t kind;   /* NG_DIST_* */
    int32_t pad;
    double a, b, lo, hi;
} ng_dist;

typedef struct {
    uint64_t steps;              /* steps simulated since ng_create                                 */
    uint64_t spikes;             /* spikes emitted                                                   */
    uint64_t events;             /* synaptic events delivered = sum over spikes of the out-degree    */
    uint64_t recorded_dropped;   /* spikes not recorded because the record was full                  */
    int64_t n_neurons;           /* neurons this handle owns (all of them on one GPU)                */
    int64_t n_connections;       /* S, connections stored on this handle                             */
    int64_t n_records_padded;    /* records stored (rows padded to a multiple of 4)                  */
    int64_t max_row_records;     /* longest padded row                                               */
    double build_ms;             /* device time of the connection build                              */
    double ms_update;            /* with NG_OPT_PROFILE: summed device time of the update kernel     */
    double ms_deliver;           /* with NG_OPT_PROFILE: summed device time of the delivery kernel   */
    uint64_t launches_update;    /* kernel launches (or graph kernel nodes executed) since create    */
    uint64_t launches_deliver;
    uint64_t launches_other;     /* builder and bookkeeping kernels                                  */
    int32_t delivery_kernel;     /* the delivery kernel in use (1 .. 6)                           */
    int32_t step_mode;
    int64_t n_sources;           /* neurons of the whole network (= n_neurons unless target-sharded)  */
    int32_t shard_rank, shard_world;   /* ng_set_shard (0, 1 on one GPU)                             */
    int32_t id_first;            /* global id of this shard's first neuron                           */
    int32_t step_kernel;         /* persistent kernel of the last ng_simulate call in step mode 2: 0 = none / two-phase
                                    (persistent_kernel<k>), 1 = persistent_pipe_kernel, 2 = the same with the spike decisions in
                                    the barrier shadow, 3 = persistent_split_kernel (list / plane barriers, decoupled warp groups) */
} ng_stats;

/* Create a simulator on cfg->device.  `alloc` may be NULL.  `cuda_stream` is a cudaStream_t (or NULL).
 * Errors: INVALID_ARG (dt <= 0, ring_slots outside 1..255, out == NULL), CUDA. */
int32_t ng_create(const ng_config* cfg, const ng_allocator* alloc, void* cuda_stream, ng_sim** out);

/* Release every device allocation and the handle.  NULL is accepted. */
int32_t ng_destroy(ng_sim* sim);

/* Message for the last error on this handle ("" if none).  Never NULL. */
const char* ng_last_error(const ng_sim* sim);

/* Add n neurons sharing one parameter set (PAPER.md:39-48 `Create`, `SetStatus`).  first_id_out (nullable)
 * receives the id of the first one.  Initial state: V = E_L, I_syn = 0, not refractory.
 * Errors: STATE after ng_prepare; INVALID_ARG for n <= 0, more than 255 populations, non-positive C_m /
 * tau_m / tau_syn / dt, |tau_m - tau_syn| < 1e-9 ms (C19), Poisson rate*h too large for the
 * 64-entry integer CDF table. */
int32_t ng_create_population(ng_sim* sim, int32_t n, const ng_lif_params* params, int32_t* first_id_out);

/* PAPER.md:37 rule "fixed indegree": every target in [tgt_first, tgt_first+tgt_n) receives exactly K
 * connections whose sources are drawn uniformly with replacement from [src_first, src_first+src_n)
 * (autapses and multapses allowed, C3).  Draw (target i, k) of call c is a pure function of
 * (seed, c, i, k) (C1-C5); call order defines c.  Nothing is built until ng_prepare.
 * Errors: STATE after ng_prepare; INVALID_ARG for ranges outside the created neurons, K < 0, bad dist. */
int32_t ng_connect_fixed_indegree(ng_sim* sim, int32_t src_first, int32_t src_n, int32_t tgt_first,
                                  int32_t tgt_n, int32_t K, const ng_dist* weight, const ng_dist* delay_steps);

/* PAPER.md:37 rule "fixed outdegree": every source sends exactly K connections to targets drawn uniformly
 * with replacement; draw (source j, k).  Same errors. */
int32_t ng_connect_fixed_outdegree(ng_sim* sim, int32_t src_first, int32_t src_n, int32_t tgt_first,
                                   int32_t tgt_n, int32_t K, const ng_dist* weight, const ng_dist* delay_steps);

/* Same rules with an explicit receptor port of the targets (0 or 1; see "Receptor ports" above).  The plain calls use
 * port 0.  Errors as above, INVALID_ARG for another port. */
int32_t ng_connect_fixed_indegree_port(ng_sim* sim, int32_t src_first, int32_t src_n, int32_t tgt_first, int32_t tgt_n,
                                       int32_t K, const ng_dist* weight, const ng_dist* delay_steps, int32_t port);
int32_t ng_connect_fixed_outdegree_port(ng_sim* sim, int32_t src_first, int32_t src_n, int32_t tgt_first, int32_t tgt_n,
                                        int32_t K, const ng_dist* weight, const ng_dist* delay_steps, int32_t port);

/* Add n AdEx neurons (Eqs. (3)-(5), alpha conductances, adaptive 5th-order Runge-Kutta).
 * Initial state: V = E_L, w = 0, conductances 0.  Errors: STATE after ng_prepare; INVALID_ARG for non-positive
 * C_m, g_L, Delta_T, tau_w, tau_syn, h_min or tolerances, too many populations, Poisson rate*h too large. */
int32_t ng_create_population_adex(ng_sim* sim, int32_t n, const ng_adex_params* params, int32_t* first_id_out);

/* Target-sharded multi-GPU (spikes of remote neurons arrive through "a spike
 * buffer, similar to the local one").  One process (or handle) per GPU; all of them issue the SAME populations and
 * connect calls with the same seed.  Handle `rank` of `world` owns the contiguous id range ng_shard_range gives: it keeps
 * the state and the input planes of those neurons and every connection whose TARGET is one of them — because a draw is a
 * pure function of (seed, call, endpoint, k), that is exactly the one-GPU structure restricted to those targets.  Each
 * time step ends its update with ONE exchange: every rank stores the ids of its spikes into the receive buffer of every
 * peer (peer-mapped device memory, NVLink) and appends what the peers stored in its own; delivery is local.
 *   ng_shard_range     pure host arithmetic (no device): first = floor(n * rank / world), n = floor(n * (rank+1) / world) - first.
 *   ng_set_shard       before ng_prepare; world 1..16.
 *   ng_exchange_handle after ng_prepare: the CUDA IPC handle (64 bytes) and/or the device pointer of this handle's receive
 *                      buffer, to be handed to the peers (the harness moves the 64 bytes with torch.distributed).
 *   ng_exchange_attach map a peer's receive buffer: its IPC handle (another process) or its pointer (same process).
 *                      Every peer must be attached before ng_simulate.
 *   ng_shard_phase     one time step in two halves — 0: update + publish, 1: gather + deliver — so that several shards that
 *                      share ONE GPU and ONE stream can be stepped without any kernel waiting for another (all phase 0
 *                      calls, then all phase 1 calls); ng_simulate does both halves per step and, on separate GPUs,
 *                      the gather kernel waits (bounded) for the peers' flags.
 * In sharded mode ng_get_state / ng_set_state address the handle's OWN neurons (element i = neuron id_first + i), stored
 * targets (ng_copy_records) are local indices, ng_get_spikes / ng_get_last_spikes / ng_stats.spikes cover the whole network
 * (global ids; every rank records all spikes), ng_stats.events and n_connections this handle's share; delivery kernel 3, step mode 2 and the statistics are one-GPU only.
 * Errors: INVALID_ARG, STATE, CUDA (a peer's list did not arrive: ng_simulate). */
int32_t ng_shard_range(int32_t n_neurons, int32_t rank, int32_t world, int32_t* first_out, int32_t* n_out);
int32_t ng_set_shard(ng_sim* sim, int32_t rank, int32_t world);
int32_t ng_exchange_handle(ng_sim* sim, void* ipc_handle_out_64, void** local_ptr_out);
int32_t ng_exchange_attach(ng_sim* sim, int32_t peer_rank, const void* ipc_handle_64, void* same_process_ptr);
int32_t ng_shard_phase(ng_sim* sim, int32_t phase);

/* Delivery-only mode (BASELINE.json configs[3], C8): the neuron update is bypassed and source s
 * fires in step n iff Philox(INJECT; s, n).x0 < floor(fraction * 2^32).  Before ng_prepare only. */
int32_t ng_set_bypass(ng_sim* sim, int32_t bypass, double inject_fraction);

/* Tuning / instrumentation knobs (NG_OPT_*).  Errors: INVALID_ARG, STATE. */
int32_t ng_set_option(ng_sim* sim, int32_t option, int64_t value);

/* Build the connection structure on the device (source-major rows, each ordered into groups of equal
 * delay, PAPER.md:69 / Fig. 1a) and allocate state.  Implied by the first ng_simulate.
 * Errors: OOM, CUDA, OVERFLOW (a drawn delay outside [1, ring_slots]); STATE if no population exists. */
int32_t ng_prepare(ng_sim* sim);

/* Copy `count` elements of a state field starting at element `first` from/to `data` (host or device).
 * Element types and lengths are listed at NG_FIELD_*.  Synchronises the stream.
 * Errors: STATE before ng_prepare; INVALID_ARG for a bad field or range. */
int32_t ng_set_state(ng_sim* sim, int32_t field, const void* data, int64_t count, int64_t first);
int32_t ng_get_state(ng_sim* sim, int32_t field, void* out, int64_t count, int64_t first);

/* Advance n_steps time steps (a1 -> a2 -> a3 each step).  Synchronises the stream before returning unless
 * NG_OPT_ASYNC is set.  Returns OVERFLOW if the spike record filled up during the call (the simulation
 * state stays valid; only recording stopped). */
int32_t ng_simulate(ng_sim* sim, int64_t n_steps);

/* Copy up to `capacity` recorded spikes (ordered by step; ids unordered within a step) into caller HOST
 * arrays and drain what was copied.  count_out always receives the number currently recorded BEFORE the
 * copy, so a call with capacity 0 sizes the buffers.  Errors: STATE (recording not enabled). */
int32_t ng_get_spikes(ng_sim* sim, int32_t* steps_host, int32_t* ids_host, int64_t capacity, int64_t* count_out);

/* Ids that spiked in the most recent step (the spike array of PAPER.md:69), into a HOST array. */
int32_t ng_get_last_spikes(ng_sim* sim, int32_t* ids_host, int64_t capacity, int64_t* count_out);

/* Connection structure read-back for parity checks (host or device destinations, any may be NULL).
 *   ng_copy_row_offsets: int64[N+1]; row j holds records [off[j], off[j+1]), padded to a multiple of 4
 *                        with records whose target is -1.
 *   ng_copy_group_offsets: uint32[N*(D+1)]; group of delay d (1-based) of source j is records
 *                        off[j] + g[j*(D+1)+d-1] .. off[j] + g[j*(D+1)+d]  (exclusive).
 *   ng_copy_records: records [first, first+count): int32 target, float weight, uint8 delay. */
int32_t ng_copy_row_offsets(ng_sim* sim, int64_t* out);
int32_t ng_copy_group_offsets(ng_sim* sim, uint32_t* out);
int32_t ng_copy_records(ng_sim* sim, int64_t first, int64_t count, int32_t* tgt, float* w, uint8_t* delay);

/* Outgoing connections of one source into HOST arrays (padding removed); count_out = its out-degree. */
int32_t ng_get_connections(ng_sim* sim, int32_t src_id, int32_t* tgt_host, float* w_host, uint8_t* delay_host,
                           int64_t capacity, int64_t* count_out);

/* Counters and timings.  Synchronises the stream. */
int32_t ng_get_stats(ng_sim* sim, ng_stats* out);

/* On-device spike statistics, the three quantities the paper validates its simulations with: per
 * neuron the average firing rate and the coefficient of variation of the inter-spike interval (standard deviation over
 * mean), and per population the Pearson correlation matrix of the spike trains of a sample of neurons re-binned to
 * bin_steps time steps (the paper: 200 neurons, 2 ms).  Accumulated at spike time inside the step kernels from
 * start_step on (the paper discards the first second); no spike record or host round trip is needed.
 *   ng_enable_statistics: after ng_prepare, once.  The sample of a population is its first sample_per_pop neurons.
 *     Spikes in bins >= max_bins are not binned (rates and CVs still count them).
 *   ng_get_rate_cv: rate_hz[N], cv_isi[N] (NaN with fewer than two intervals) into host or device arrays.
 *   ng_get_correlations: corr[ns*ns] row-major over the complete bins so far (NaN for a silent train); n_sample_out = ns
 *     and n_bins_out are always set, the matrix is written only if capacity >= ns*ns.
 * Errors: STATE (before ng_prepare, not enabled, enabled twice, nothing simulated yet), INVALID_ARG, OOM. */
int32_t ng_enable_statistics(ng_sim* sim, int64_t start_step, int32_t bin_steps, int32_t sample_per_pop, int32_t max_bins);
int32_t ng_get_rate_cv(ng_sim* sim, float* rate_hz, float* cv_isi, int64_t count);
int32_t ng_get_correlations(ng_sim* sim, int32_t population, float* corr, int64_t capacity, int32_t* n_sample_out,
                            int32_t* n_bins_out);

/* Phase stamps of the last persistent launch (NG_OPT_TRACE): uint64 ns (%globaltimer), laid out
 * [64 steps][blocks][16 stamps], step index = step mod 64, one stamping thread per CTA and stamp.
 *   two-phase kernels (delivery kernel 1, 2): 0 step start, 1 update done, 2 after the first barrier, 3 delivery done,
 *     5 after the second barrier;
 *   pipelined kernel (3): 0 phase start, 3 update done (warp 0), 4 all updater warps done, 6 delay-1 pass done,
 *     7 rest pass: spike count known, 8 rest pass: entries staged, 9 rest pass: items done, 1 phase done, 2 after the barrier.
 * count_out = words available, blocks_out = CTAs of that launch; copies only if capacity >= count.
 * Errors: STATE when no trace exists. */
int32_t ng_get_trace(ng_sim* sim, uint64_t* out_host, int64_t capacity, int64_t* count_out, int32_t* blocks_out);

/* Ceiling probe for the roofline report (not on the hot path).  Measures, with the load and
 * reduction instructions the delivery kernels use, what this GPU sustains for
 *   kind 0: a coalesced 128-bit read stream over 2 GiB                        -> bytes per second
 *   kind 1: red.global.add.f32 to uniformly random cells of a footprint_bytes array -> reductions per second
 *   kind 2: streamed 8-byte records + one random reduction per record (the shape of a3) -> events per second
 * Allocates its own scratch with cudaMalloc and frees it.  Errors: INVALID_ARG, OOM, CUDA. */
int32_t ng_probe(int32_t device, int32_t kind, int64_t footprint_bytes, double* per_second_out);

/* ---- Spike delivery that allocates nothing (csrc/ng_noalloc.cu) --------------------------------------------------
 * For callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it.  One step n of a3 (every connection (j -> i, w, d) of a neuron j that spiked in step n adds w to
 * ring slot (n + d) mod D of target i) on caller-owned DEVICE arrays, with the ring — the only scratch the step
 * needs — in a static device array of the library instead of allocated memory:
 *     NG_NOALLOC_MAX_CELLS = 4,194,304 float cells = 16 MiB, held by every GPU that loads libng.so until exit;
 *     n_targets * ring_slots beyond it is rejected with NG_ERR_INVALID_ARG (use ng_create / ng_simulate there).
 * What one call does, in stream order on cuda_stream (NULL = legacy default stream) of the CURRENT device:
 *     reset != 0: the ring is cleared first (the array keeps the last call's contents: pass reset on the first call
 *                 of a sequence, and whenever the network or the step sequence changes);
 *     input_out_dev[i] = ring[(step mod D) * n_targets + i], i < n_targets — the input arriving at step n, what
 *                 the neuron update of step n consumes (NG_FIELD_LAST_INPUT) — and that plane is cleared;
 *     for every s < n_spikes, j = spike_ids_dev[s], every record r in [row_offsets_dev[j], row_offsets_dev[j+1]):
 *                 ring[((step + delay_dev[r]) mod D) * n_targets + tgt_dev[r]] += w_dev[r]   (red.global.add.f32).
 * The connection arrays have the layout ng_copy_row_offsets / ng_copy_records return (source-major rows, int64
 * offsets [n_sources + 1], records with tgt < 0 are padding and skipped); rows that start and end on multiples of
 * 4 records in 16-byte aligned arrays are read with 128-bit loads, any other layout with scalar loads.  A record whose
 * target is >= n_targets or whose delay is outside [1, ring_slots], and a spike id outside [0, n_sources), is
 * skipped and counted; ng_deliver_noalloc_check synchronises the stream, returns the count since the last check
 * (n_bad_out may be NULL) and NG_ERR_OVERFLOW if it is not zero.
 * The call enqueues two kernels (and one memset with reset) and returns without synchronising; it calls no
 * cudaMalloc, cudaFree or allocating library routine.  Ownership: all arrays stay the caller's.
 * ALL calls on one GPU share the one static ring: calls that overlap on the GPU (two streams, two host threads, two
 * simulations interleaved step by step) race on it — one sequence of steps at a time per GPU.
 * Errors: INVALID_ARG (sizes, NULL arrays), CUDA.  ng_noalloc_last_error() gives the message of the calling
 * thread's last failing ng_deliver_noalloc* call ("" if none). */
#define NG_NOALLOC_MAX_CELLS (1 << 22)
int32_t ng_deliver_noalloc(void* cuda_stream, const int64_t* row_offsets_dev, const int32_t* tgt_dev, const float* w_dev,
                           const uint8_t* delay_dev, int32_t n_sources, const int32_t* spike_ids_dev, int32_t n_spikes,
                           int32_t n_targets, int32_t ring_slots, int64_t step, int32_t reset, float* input_out_dev);
int32_t ng_deliver_noalloc_check(void* cuda_stream, int64_t* n_bad_out);
const char* ng_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* NG_H_ */
