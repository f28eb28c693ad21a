// =====================================================================================
// oracle.cpp — TEST INFRASTRUCTURE. NOT part of the product path.
//
// A plain, slow, single-threaded fp64 CPU restatement of the per-time-step hot path of a
// clock-driven spiking-network simulator as arXiv 2007.14236 defines it, plus
// the seeded connection builder that feeds it.  It shares no code, header, table or
// constant generator with the CUDA path under paper_2007_14236_b200/csrc/ and neither
// includes the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference leg may load it.
//
// What it follows (PAPER.md line : passage):
//   93-97  Eq. (1)  tau_m dV/dt = -(V - E_L) + R_m I_syn                (LIF membrane)
//   97-102 Eq. (2)  tau_syn dI/dt = -I + sum_j w_ij sum_f delta(t-t_j^f) (exponential PSC;
//                   printed sum index is garbled — DESIGN.md reading C13: sum over
//                   presynaptic j, a spike raises I by w)
//   37     "integrated by the exact integration scheme described in [20] on the time grid"
//          (Rotter & Diesmann 1999: propagator matrix exp(A h) of the linear system)
//   69     spike-delivery: a spike of a source reaches the connection group of delay d
//          when its time index matches d                                (delay semantics)
//   187    refractory time 2 ms;  181  time step 0.1 ms
// Where the paper is silent the readings C1..C20 of DESIGN.md apply (RNG contract, delay
// rounding, Poisson drive, threshold/reset order).
//
// Delivery reaches exactly its plain definition:
//     in_i(n) = sum over connections c with tgt(c)=i of  w_c * S_src(c)(n - d_c)
// The stepper below realises it push-style through a D-slot ring exactly in the order the
// DESIGN.md algorithm states; tests/ additionally brute-force the plain definition with a
// dense W[d][i][j] and a spike-history matrix on networks of <= 50 neurons.
//
// Pins (tests/test_oracle_*.py, all run with -m "not gpu"):
//   philox        — published known-answer vectors (Salmon et al., SC'11, Random123 KAT)
//   propagators   — scipy.linalg.expm of the system matrix; semigroup identity
//   PSP response  — analytic solution of Eqs. (1)-(2) at grid points, peak 0.15 mV
//   refractoriness— closed-form grid ISI for constant supra-threshold current
//   poisson       — scipy.stats.poisson CDF, sample mean/variance, Campbell's theorem
//   connectivity  — exact in-degree per call, uniform/normal statistics vs scipy.stats
//   delivery      — dense brute force (numpy) and per-step weight-sum invariants
//   free-running network activity: "parity unpinned" beyond the above (paper prints no rates)
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>

#include "oracle_adex.hpp"

namespace {

// ---------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as
// 1, 2, 3", SC'11).  DESIGN.md reading C1: key = 64-bit seed (lo, hi), counter = 4 x u32.
// ---------------------------------------------------------------------------------
void philox4x32_10(uint32_t key_lo, uint32_t key_hi, const uint32_t ctr[4], uint32_t out[4]) {
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;      // round multipliers
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;      // Weyl key increments
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key_lo, k1 = key_hi;
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += W0; k1 += W1; }
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum { TAG_CONN = 1, TAG_POISSON = 2, TAG_INJECT = 3 };     // counter word 3 (reading C1)
enum { DIST_CONST = 0, DIST_NORMAL_CLIPPED = 1, DIST_UNIFORM_INT = 2 };
enum { RULE_FIXED_INDEGREE = 0, RULE_FIXED_OUTDEGREE = 1 };
enum { FIELD_V = 0, FIELD_I_SYN = 1, FIELD_REFR = 2, FIELD_RING = 3, FIELD_STEP = 4,
       FIELD_W = 6, FIELD_G_EX = 7, FIELD_Y_EX = 8, FIELD_G_IN = 9, FIELD_Y_IN = 10, FIELD_H_INT = 11 };   // AdEx state
enum { MODEL_LIF = 0, MODEL_ADEX = 1 };

struct LifParams {           // PAPER.md:93-102 symbols; units pF, ms, mV, pA, Hz
    double C_m, tau_m, tau_syn, E_L, V_th, V_reset, t_ref_ms, I_e, poisson_rate_hz, poisson_weight;
};
struct Dist { int32_t kind; int32_t pad; double a, b, lo, hi; };

struct Population {
    int32_t first, n;
    int32_t model = MODEL_LIF;
    adex::Params ax{};                // MODEL_ADEX (oracle_adex.hpp)
    LifParams p;
    double P11, P22, P21, P20;        // exact-integration propagators
    int32_t refr_steps;
    std::vector<uint32_t> poisson_T;  // integer CDF table (reading C7)
};
struct ConnectCall {
    int32_t rule, src_first, src_n, tgt_first, tgt_n, K;
    Dist w, d;
    int32_t port = 0;                 // receptor port of the targets: 0 excitatory (and the LIF current), 1 inhibitory
};
struct Conn { int32_t src, tgt; int32_t delay; float w; int32_t call; int32_t endpoint; int32_t k; int32_t port; };

// Exact-integration propagators of Eqs. (1)-(2) over one step h (ref. 20).
// State x = (I, V - E_L);  dx/dt = A x,  A = [[-1/tau_syn, 0], [1/C_m, -1/tau_m]]  (R_m = tau_m/C_m).
// exp(A h) = [[P11, 0], [P21, P22]];  a constant current I_e adds P20 * I_e to V.
void propagators(const LifParams& p, double h, double& P11, double& P22, double& P21, double& P20) {
    P11 = std::exp(-h / p.tau_syn);
    P22 = std::exp(-h / p.tau_m);
    P21 = p.tau_m * p.tau_syn / (p.C_m * (p.tau_m - p.tau_syn)) * (P22 - P11);
    P20 = p.tau_m / p.C_m * (1.0 - P22);
}

// Reading C7: T[m] = floor(CDF_Poisson(lam)(m) * 2^32), saturating; count k = #{m : x >= T[m]}.
int poisson_table(double lam, std::vector<uint32_t>& T) {
    T.clear();
    if (!(lam > 0.0)) return 0;
    double p = std::exp(-lam);
    double c = p;
    for (int m = 0; m < 64; ++m) {
        double s = std::floor(c * 4294967296.0);
        uint32_t t = (s >= 4294967295.0) ? 4294967295u : (uint32_t)s;
        T.push_back(t);
        if (t == 4294967295u) return 0;
        double pl = p * lam;
        p = pl / (double)(m + 1);
        c = c + p;
    }
    return -1;   // lam too large for a 64-entry table
}

struct Sim {
    double dt_ms; int32_t D; uint64_t seed;
    int32_t bypass_neurons = 0; uint32_t inject_thr = 0;
    std::vector<Population> pops;
    std::vector<ConnectCall> calls;
    int32_t N = 0;
    bool prepared = false;
    // canonical connection list, ordered by (src, delay, tgt, call, k)   (reading C18)
    std::vector<Conn> conns;
    std::vector<int64_t> row_off;          // N+1
    // state (fp64)
    std::vector<double> V, I; std::vector<int32_t> refr; std::vector<int32_t> pop_of;
    std::vector<double> ring;              // [D][P][N], slot-major, P = n_ports
    int32_t P = 1;                         // receptor ports: 2 as soon as an AdEx population exists
    std::vector<adex::State> ax;           // AdEx state (unused entries for LIF neurons)
    int64_t step = 0;
    std::vector<int32_t> spk_step, spk_id; // spike record
    std::vector<int32_t> last_spikes;      // ids that spiked in the most recent step
    uint64_t events = 0;
    std::string err;
};

// One connection draw, O(1) from (call, endpoint, k)  — readings C1-C5.
void draw_conn(const Sim& s, int32_t call_idx, int32_t endpoint, int32_t k, Conn& out) {
    const ConnectCall& c = s.calls[call_idx];
    uint32_t ctr[4] = {(uint32_t)k, (uint32_t)endpoint, (uint32_t)call_idx, (uint32_t)TAG_CONN};
    uint32_t x[4];
    philox4x32_10((uint32_t)s.seed, (uint32_t)(s.seed >> 32), ctr, x);
    // C2: other end by multiply-high range reduction
    if (c.rule == RULE_FIXED_INDEGREE) {
        out.tgt = endpoint;
        out.src = c.src_first + (int32_t)(((uint64_t)x[0] * (uint64_t)(uint32_t)c.src_n) >> 32);
    } else {
        out.src = endpoint;
        out.tgt = c.tgt_first + (int32_t)(((uint64_t)x[0] * (uint64_t)(uint32_t)c.tgt_n) >> 32);
    }
    // C4: Box-Muller pair in fp64 from (x1, x2)
    double z_w = 0.0, z_d = 0.0;
    if (c.w.kind == DIST_NORMAL_CLIPPED || c.d.kind == DIST_NORMAL_CLIPPED) {
        double u1 = ((double)x[1] + 0.5) * (1.0 / 4294967296.0);
        double u2 = ((double)x[2] + 0.5) * (1.0 / 4294967296.0);
        double r = std::sqrt(-2.0 * std::log(u1));
        double a = 6.283185307179586476925286766559 * u2;
        z_w = r * std::cos(a);
        z_d = r * std::sin(a);
    }
    // weight: fp32 quantity (the connection record stores fp32)
    double w;
    if (c.w.kind == DIST_CONST) w = c.w.a;
    else if (c.w.kind == DIST_NORMAL_CLIPPED) {
        double t = c.w.b * z_w;
        w = c.w.a + t;
        if (w < c.w.lo) w = c.w.lo;
        if (w > c.w.hi) w = c.w.hi;
    } else {  // uniform int as a weight: not used by any config; defined for completeness
        double span = c.w.hi - c.w.lo + 1.0;
        w = c.w.lo + (double)(((uint64_t)x[3] * (uint64_t)span) >> 32);
    }
    out.w = (float)w;
    // delay in steps, C5
    int64_t d;
    if (c.d.kind == DIST_CONST) d = (int64_t)c.d.a;
    else if (c.d.kind == DIST_UNIFORM_INT) {
        uint64_t span = (uint64_t)((int64_t)c.d.hi - (int64_t)c.d.lo + 1);
        d = (int64_t)c.d.lo + (int64_t)(((uint64_t)x[3] * span) >> 32);
    } else {
        double t = c.d.b * z_d;
        double v = c.d.a + t;
        double f = std::floor(v + 0.5);
        if (f < c.d.lo) f = c.d.lo;
        if (f > c.d.hi) f = c.d.hi;
        d = (int64_t)f;
    }
    out.delay = (int32_t)d;
    out.call = call_idx; out.endpoint = endpoint; out.k = k; out.port = c.port;
}

int poisson_count(const Sim& s, const Population& pop, int32_t i, int64_t n) {
    if (pop.poisson_T.empty()) return 0;
    uint32_t ctr[4] = {(uint32_t)i, (uint32_t)((uint64_t)n & 0xffffffffu), (uint32_t)((uint64_t)n >> 32),
                       (uint32_t)TAG_POISSON};
    uint32_t x[4];
    philox4x32_10((uint32_t)s.seed, (uint32_t)(s.seed >> 32), ctr, x);
    int k = 0;
    for (uint32_t t : pop.poisson_T) if (x[0] >= t) ++k;
    return k;
}

bool inject_fires(const Sim& s, int32_t i, int64_t n) {   // reading C8
    uint32_t ctr[4] = {(uint32_t)i, (uint32_t)((uint64_t)n & 0xffffffffu), (uint32_t)((uint64_t)n >> 32),
                       (uint32_t)TAG_INJECT};
    uint32_t x[4];
    philox4x32_10((uint32_t)s.seed, (uint32_t)(s.seed >> 32), ctr, x);
    return x[0] < s.inject_thr;
}

int prepare(Sim& s) {
    if (s.prepared) return 0;
    s.N = 0;
    for (auto& p : s.pops) s.N += p.n;
    const int32_t N = s.N;
    // 1. draw every connection in call order, endpoint ascending, k ascending
    s.conns.clear();
    size_t total = 0;                     // storage only: one allocation instead of doubling (1e9 records at config 4)
    for (const ConnectCall& c : s.calls) total += (size_t)((c.rule == RULE_FIXED_INDEGREE) ? c.tgt_n : c.src_n) * (size_t)c.K;
    s.conns.reserve(total);
    for (int32_t ci = 0; ci < (int32_t)s.calls.size(); ++ci) {
        const ConnectCall& c = s.calls[ci];
        int32_t e_first = (c.rule == RULE_FIXED_INDEGREE) ? c.tgt_first : c.src_first;
        int32_t e_n = (c.rule == RULE_FIXED_INDEGREE) ? c.tgt_n : c.src_n;
        for (int32_t e = e_first; e < e_first + e_n; ++e)
            for (int32_t k = 0; k < c.K; ++k) {
                Conn cn; draw_conn(s, ci, e, k, cn);
                if (cn.delay < 1 || cn.delay > s.D) { s.err = "delay outside [1, D]"; return -5; }
                s.conns.push_back(cn);
            }
    }
    // 2. canonical order (src, delay, tgt, call, k)
    std::sort(s.conns.begin(), s.conns.end(), [](const Conn& a, const Conn& b) {
        if (a.src != b.src) return a.src < b.src;
        if (a.delay != b.delay) return a.delay < b.delay;
        if (a.tgt != b.tgt) return a.tgt < b.tgt;
        if (a.call != b.call) return a.call < b.call;
        if (a.endpoint != b.endpoint) return a.endpoint < b.endpoint;
        return a.k < b.k;
    });
    s.row_off.assign((size_t)N + 1, 0);
    for (const Conn& c : s.conns) s.row_off[(size_t)c.src + 1]++;
    for (int32_t i = 0; i < N; ++i) s.row_off[(size_t)i + 1] += s.row_off[i];
    // 3. state
    s.V.assign(N, 0.0); s.I.assign(N, 0.0); s.refr.assign(N, 0); s.pop_of.assign(N, 0);
    for (int32_t pi = 0; pi < (int32_t)s.pops.size(); ++pi) {
        Population& p = s.pops[pi];
        for (int32_t i = p.first; i < p.first + p.n; ++i) { s.V[i] = p.p.E_L; s.pop_of[i] = pi; }
    }
    s.P = 1;
    for (auto& p : s.pops) if (p.model == MODEL_ADEX) s.P = 2;
    s.ax.assign(N, adex::State{});
    for (auto& p : s.pops) if (p.model == MODEL_ADEX)
        for (int32_t i = p.first; i < p.first + p.n; ++i) {
            adex::State st{}; st.y[0] = p.ax.E_L; st.h_int = s.dt_ms;
            s.ax[i] = st; s.V[i] = p.ax.E_L;
        }
    s.ring.assign((size_t)s.D * (size_t)s.P * (size_t)N, 0.0);
    s.step = 0;
    s.prepared = true;
    return 0;
}

// One time step n: t_n -> t_{n+1}.  DESIGN.md oracle algorithm, steps 3a-3d then 4.
void step_once(Sim& s, bool record) {
    const int32_t N = s.N; const int32_t D = s.D; const int64_t n = s.step;
    const size_t P = (size_t)s.P;
    const size_t slot = (size_t)(n % D);
    s.last_spikes.clear();
    for (int32_t i = 0; i < N; ++i) {
        // 3a. consume and clear this step's ring slot (port 0; port 1 exists only next to AdEx populations)
        double in = s.ring[(slot * P) * N + i];
        s.ring[(slot * P) * N + i] = 0.0;
        double in1 = 0.0;
        if (P > 1) { in1 = s.ring[(slot * P + 1) * N + i]; s.ring[(slot * P + 1) * N + i] = 0.0; }
        if (s.bypass_neurons) {                       // config-3 mode, reading C8
            if (inject_fires(s, i, n)) s.last_spikes.push_back(i);
            continue;
        }
        const Population& pop = s.pops[s.pop_of[i]];
        int k = poisson_count(s, pop, i, n);
        if (pop.model == MODEL_ADEX) {
            // AdEx + alpha conductances, adaptive RK5 over the step (oracle_adex.hpp), then the
            // conductance jumps arriving at t_{n+1} (C25): y += W e / tau for both ports, Poisson drive on port 0
            adex::State& st = s.ax[i];
            st.y[0] = s.V[i];
            const bool spk = adex::step(pop.ax, st, s.dt_ms);
            const double jump = std::exp(1.0) / pop.ax.tau_syn;
            st.y[3] += jump * (in + pop.ax.poisson_weight * (double)k);
            st.y[5] += jump * in1;
            s.V[i] = st.y[0];
            if (spk) s.last_spikes.push_back(i);
            continue;
        }
        // 3b. membrane: exact integration with the current *before* its update (C11)
        if (s.refr[i] == 0) {
            s.V[i] = pop.p.E_L + pop.P22 * (s.V[i] - pop.p.E_L) + pop.P21 * s.I[i] + pop.P20 * pop.p.I_e;
        } else {
            s.refr[i] -= 1;
        }
        // 3c. synaptic current: decay, then the jumps arriving at t_{n+1} (C10, C13) and the drive (C7)
        s.I[i] = pop.P11 * s.I[i] + in + pop.p.poisson_weight * (double)k;
        // 3d. threshold, reset, refractoriness (C11)
        if (s.V[i] >= pop.p.V_th) {
            s.last_spikes.push_back(i);
            s.V[i] = pop.p.V_reset;
            s.refr[i] = pop.refr_steps;
        }
    }
    // 4. delivery: every outgoing connection (j -> i, w, d) of a spiking j adds w to slot (n + d) mod D
    for (int32_t j : s.last_spikes) {
        if (record) { s.spk_step.push_back((int32_t)n); s.spk_id.push_back(j); }
        for (int64_t c = s.row_off[j]; c < s.row_off[(size_t)j + 1]; ++c) {
            const Conn& cn = s.conns[(size_t)c];
            size_t sl = (size_t)((n + cn.delay) % D);
            s.ring[(sl * P + (size_t)cn.port) * N + cn.tgt] += (double)cn.w;
        }
        s.events += (uint64_t)(s.row_off[(size_t)j + 1] - s.row_off[j]);
    }
    s.step = n + 1;
}

}  // namespace

// ---------------------------------------------------------------------------------
// C interface for the Python test harness (ctypes).  Names are orc_*, distinct from the
// product's ng_* C-ABI; nothing here is declared in include/.
// ---------------------------------------------------------------------------------
extern "C" {

void orc_philox4x32_10(uint32_t key_lo, uint32_t key_hi, const uint32_t* ctr, uint32_t* out) {
    philox4x32_10(key_lo, key_hi, ctr, out);
}

void orc_propagators(const LifParams* p, double h, double* out4) {
    propagators(*p, h, out4[0], out4[1], out4[2], out4[3]);
}

int32_t orc_poisson_table(double lam, uint32_t* out, int32_t cap) {
    std::vector<uint32_t> T;
    if (poisson_table(lam, T) != 0) return -1;
    for (int32_t i = 0; i < (int32_t)T.size() && i < cap; ++i) out[i] = T[i];
    return (int32_t)T.size();
}

void* orc_create(double dt_ms, int32_t D, uint64_t seed) {
    Sim* s = new Sim();
    s->dt_ms = dt_ms; s->D = D; s->seed = seed;
    return s;
}
void orc_destroy(void* h) { delete (Sim*)h; }
const char* orc_last_error(void* h) { return ((Sim*)h)->err.c_str(); }

int32_t orc_set_bypass(void* h, int32_t bypass, double inject_fraction) {
    Sim* s = (Sim*)h;
    s->bypass_neurons = bypass;
    double t = std::floor(inject_fraction * 4294967296.0);
    if (t < 0.0) t = 0.0;
    if (t > 4294967295.0) t = 4294967295.0;
    s->inject_thr = (uint32_t)t;
    return 0;
}

int32_t orc_create_population(void* h, int32_t n, const LifParams* p, int32_t* first_out) {
    Sim* s = (Sim*)h;
    if (s->prepared) { s->err = "population after prepare"; return -2; }
    if (n <= 0) { s->err = "n <= 0"; return -1; }
    if (std::fabs(p->tau_m - p->tau_syn) < 1e-9) { s->err = "tau_m == tau_syn"; return -1; }   // C19
    Population pop;
    pop.first = s->N; pop.n = n; pop.p = *p;
    propagators(*p, s->dt_ms, pop.P11, pop.P22, pop.P21, pop.P20);
    pop.refr_steps = (int32_t)std::floor(p->t_ref_ms / s->dt_ms + 0.5);
    double lam = p->poisson_rate_hz * s->dt_ms * 1e-3;
    if (poisson_table(lam, pop.poisson_T) != 0) { s->err = "poisson rate too large"; return -1; }
    s->pops.push_back(pop);
    s->N += n;
    if (first_out) *first_out = pop.first;
    return 0;
}

int32_t orc_connect_port(void* h, int32_t rule, int32_t src_first, int32_t src_n, int32_t tgt_first, int32_t tgt_n,
                         int32_t K, const Dist* w, const Dist* d, int32_t port) {
    Sim* s = (Sim*)h;
    if (s->prepared) { s->err = "connect after prepare"; return -2; }
    if (src_n <= 0 || tgt_n <= 0 || K < 0 || src_first < 0 || tgt_first < 0 || port < 0 || port > 1 ||
        src_first + src_n > s->N || tgt_first + tgt_n > s->N) { s->err = "bad range"; return -1; }
    ConnectCall c{rule, src_first, src_n, tgt_first, tgt_n, K, *w, *d, port};
    s->calls.push_back(c);
    return 0;
}
int32_t orc_connect(void* h, int32_t rule, int32_t src_first, int32_t src_n, int32_t tgt_first, int32_t tgt_n,
                    int32_t K, const Dist* w, const Dist* d) {
    return orc_connect_port(h, rule, src_first, src_n, tgt_first, tgt_n, K, w, d, 0);
}

int32_t orc_create_population_adex(void* h, int32_t n, const adex::Params* p, int32_t* first_out) {
    Sim* s = (Sim*)h;
    if (s->prepared) { s->err = "population after prepare"; return -2; }
    if (n <= 0) { s->err = "n <= 0"; return -1; }
    Population pop;
    pop.first = s->N; pop.n = n; pop.model = MODEL_ADEX; pop.ax = *p; pop.p = LifParams{};
    pop.P11 = pop.P22 = pop.P21 = pop.P20 = 0.0; pop.refr_steps = 0;
    double lam = p->poisson_rate_hz * s->dt_ms * 1e-3;
    if (poisson_table(lam, pop.poisson_T) != 0) { s->err = "poisson rate too large"; return -1; }
    s->pops.push_back(pop);
    s->N += n;
    if (first_out) *first_out = pop.first;
    return 0;
}

// single-neuron helpers for the pins: the right-hand side and one time step of the AdEx integrator
void orc_adex_rhs(const adex::Params* p, const double* y6, double* f6) { adex::rhs(*p, y6, f6); }
int32_t orc_adex_step(const adex::Params* p, double* y6, double* h_int, double h_step) {
    adex::State st; for (int i = 0; i < 6; ++i) st.y[i] = y6[i]; st.h_int = *h_int;
    const bool spk = adex::step(*p, st, h_step);
    for (int i = 0; i < 6; ++i) y6[i] = st.y[i]; *h_int = st.h_int;
    return spk ? 1 : 0;
}
int32_t orc_num_ports(void* h) { return ((Sim*)h)->P; }

int32_t orc_prepare(void* h) { return prepare(*(Sim*)h); }

int64_t orc_num_connections(void* h) { return (int64_t)((Sim*)h)->conns.size(); }
int32_t orc_num_neurons(void* h) { return ((Sim*)h)->N; }

// Canonical COO + row offsets.  Any output pointer may be null.
int32_t orc_get_connections(void* h, int32_t* src, int32_t* tgt, float* w, uint8_t* delay, int64_t* row_off) {
    Sim* s = (Sim*)h;
    if (!s->prepared) return -2;
    for (size_t c = 0; c < s->conns.size(); ++c) {
        if (src) src[c] = s->conns[c].src;
        if (tgt) tgt[c] = s->conns[c].tgt;
        if (w) w[c] = s->conns[c].w;
        if (delay) delay[c] = (uint8_t)s->conns[c].delay;
    }
    if (row_off) for (size_t i = 0; i < s->row_off.size(); ++i) row_off[i] = s->row_off[i];
    return 0;
}

// Regenerate one draw in O(1): out = {src, tgt, delay}, *w_out = weight.
int32_t orc_draw_connection(void* h, int32_t call, int32_t endpoint, int32_t k, int32_t* out3, float* w_out) {
    Sim* s = (Sim*)h;
    if (call < 0 || call >= (int32_t)s->calls.size()) return -1;
    Conn c; draw_conn(*s, call, endpoint, k, c);
    out3[0] = c.src; out3[1] = c.tgt; out3[2] = c.delay; *w_out = c.w;
    return 0;
}

int32_t orc_poisson_count(void* h, int32_t i, int64_t n) {
    Sim* s = (Sim*)h;
    if (!s->prepared) return -2;
    return poisson_count(*s, s->pops[s->pop_of[i]], i, n);
}

int32_t orc_set_state(void* h, int32_t field, const void* data, int64_t n, int64_t first) {
    Sim* s = (Sim*)h;
    if (!s->prepared) return -2;
    if (field == FIELD_V) { for (int64_t i = 0; i < n; ++i) s->V[first + i] = ((const double*)data)[i]; }
    else if (field == FIELD_I_SYN) { for (int64_t i = 0; i < n; ++i) s->I[first + i] = ((const double*)data)[i]; }
    else if (field == FIELD_REFR) { for (int64_t i = 0; i < n; ++i) s->refr[first + i] = ((const int32_t*)data)[i]; }
    else if (field == FIELD_RING) { for (int64_t i = 0; i < n; ++i) s->ring[first + i] = ((const double*)data)[i]; }
    else if (field == FIELD_STEP) { s->step = *(const int64_t*)data; }
    else if (field >= FIELD_W && field <= FIELD_Y_IN) { for (int64_t i = 0; i < n; ++i) s->ax[first + i].y[field - FIELD_W + 1] = ((const double*)data)[i]; }
    else if (field == FIELD_H_INT) { for (int64_t i = 0; i < n; ++i) s->ax[first + i].h_int = ((const double*)data)[i]; }
    else return -1;
    return 0;
}
int32_t orc_get_state(void* h, int32_t field, void* data, int64_t n, int64_t first) {
    Sim* s = (Sim*)h;
    if (!s->prepared) return -2;
    if (field == FIELD_V) { for (int64_t i = 0; i < n; ++i) ((double*)data)[i] = s->V[first + i]; }
    else if (field == FIELD_I_SYN) { for (int64_t i = 0; i < n; ++i) ((double*)data)[i] = s->I[first + i]; }
    else if (field == FIELD_REFR) { for (int64_t i = 0; i < n; ++i) ((int32_t*)data)[i] = s->refr[first + i]; }
    else if (field == FIELD_RING) { for (int64_t i = 0; i < n; ++i) ((double*)data)[i] = s->ring[first + i]; }
    else if (field == FIELD_STEP) { *(int64_t*)data = s->step; }
    else if (field >= FIELD_W && field <= FIELD_Y_IN) { for (int64_t i = 0; i < n; ++i) ((double*)data)[i] = s->ax[first + i].y[field - FIELD_W + 1]; }
    else if (field == FIELD_H_INT) { for (int64_t i = 0; i < n; ++i) ((double*)data)[i] = s->ax[first + i].h_int; }
    else return -1;
    return 0;
}

int32_t orc_simulate(void* h, int64_t n_steps, int32_t record) {
    Sim* s = (Sim*)h;
    int rc = prepare(*s);
    if (rc) return rc;
    for (int64_t i = 0; i < n_steps; ++i) step_once(*s, record != 0);
    return 0;
}

int64_t orc_num_spikes(void* h) { return (int64_t)((Sim*)h)->spk_id.size(); }
int32_t orc_get_spikes(void* h, int32_t* steps, int32_t* ids, int64_t cap, int32_t drain) {
    Sim* s = (Sim*)h;
    int64_t n = std::min<int64_t>(cap, (int64_t)s->spk_id.size());
    for (int64_t i = 0; i < n; ++i) { steps[i] = s->spk_step[i]; ids[i] = s->spk_id[i]; }
    if (drain) { s->spk_step.clear(); s->spk_id.clear(); }
    return 0;
}
int64_t orc_num_last_spikes(void* h) { return (int64_t)((Sim*)h)->last_spikes.size(); }
void orc_get_last_spikes(void* h, int32_t* ids) {
    Sim* s = (Sim*)h;
    for (size_t i = 0; i < s->last_spikes.size(); ++i) ids[i] = s->last_spikes[i];
}
uint64_t orc_num_events(void* h) { return ((Sim*)h)->events; }

}  // extern "C"
