// =====================================================================================
// oracle_adex.hpp — TEST INFRASTRUCTURE (included by oracle.cpp only).
//
// fp64 restatement of the AdEx neuron with conductance-based alpha synapses that the paper's balanced network uses
// (PAPER.md:110-161): Eq. (3) membrane, Eq. (4) synaptic current, Eq. (5) adaptation, Table II parameters, integrated
// with "the 5th order Runge-Kutta method with adaptive control of the step size".
//
// Readings of what the paper leaves open (C21-C25):
//   C21  Eq. (4) prints I_syn = sum_i g_i (V - E_rev,i) added with a plus sign in Eq. (3); that sign would make an
//        excitatory conductance hyperpolarise.  Read as I_syn = sum_i g_i (E_rev,i - V).
//   C22  "synaptic conductance modeled by an alpha function": g' = -g/tau + y, y' = -y/tau, a spike of
//        weight W (nS) raises y by W e / tau, so the conductance peaks at W one tau after the spike.
//   C23  the Runge-Kutta pair and its controller are not named: embedded Cash-Karp 5(4), error = max_i |Delta_i| / tol_i
//        with absolute tolerances per component, h_new = 0.9 h err^(-1/5) limited to [0.2, 5] h, sub-steps clipped to the
//        end of the time step, smallest sub-step h_min accepted unconditionally; the sub-step size is neuron state.
//   C24  spike when V >= V_peak after an accepted sub-step: V <- V_r, w <- w + b; V_peak and the
//        refractory time are not in Table II: V_peak = 0 mV, t_ref = 0; one spike per neuron and time step (C20); the
//        exponential is evaluated at min(V, V_peak).
//   C25  inputs arrive on the time grid like the LIF currents (C10): the conductance jumps of step n are applied at
//        t_{n+1}, after the integration of step n; the Poisson drive goes to the excitatory port.
// Pins (tests/test_oracle_adex.py): scipy.integrate.solve_ivp (LSODA/Radau, rtol 1e-10) on the single-neuron 700 pA
// protocol of PAPER.md:252 between spikes, the closed-form alpha conductance, fixed points, spike count of that
// protocol against the event-located scipy solution.
// =====================================================================================
#pragma once
#include <algorithm>
#include <cmath>

namespace adex {

struct Params {              // Table II symbols; units pF, nS, mV, ms, pA, Hz
    double C_m, g_L, E_L, V_T, Delta_T, tau_w, a, b, V_reset, V_peak, E_ex, E_in, tau_syn, I_e;
    double poisson_rate_hz, poisson_weight;
    double tol[6];           // absolute tolerances of (V, w, g_ex, y_ex, g_in, y_in) for the step-size controller
    double h_min;            // smallest sub-step, ms
};
struct State { double y[6]; double h_int; };     // y = (V, w, g_ex, y_ex, g_in, y_in)

inline void rhs(const Params& p, const double* y, double* f) {
    const double V = std::min(y[0], p.V_peak);                                    // C24
    const double I_spike = p.g_L * p.Delta_T * std::exp((V - p.V_T) / p.Delta_T);
    const double I_syn = y[2] * (p.E_ex - V) + y[4] * (p.E_in - V);               // C21
    f[0] = (-p.g_L * (V - p.E_L) + I_spike + I_syn - y[1] + p.I_e) / p.C_m;      // Eq. (3)
    f[1] = (p.a * (V - p.E_L) - y[1]) / p.tau_w;                                  // Eq. (5)
    f[2] = -y[2] / p.tau_syn + y[3];                                              // C22
    f[3] = -y[3] / p.tau_syn;
    f[4] = -y[4] / p.tau_syn + y[5];
    f[5] = -y[5] / p.tau_syn;
}

// One Cash-Karp step of size h from y: 5th-order result in y5, error estimate (5th - 4th order) in err.
inline void cash_karp(const Params& p, const double* y, double h, double* y5, double* err) {
    static const double a2 = 0.2, b21 = 0.2;
    static const double b31 = 3.0 / 40.0, b32 = 9.0 / 40.0;
    static const double b41 = 0.3, b42 = -0.9, b43 = 1.2;
    static const double b51 = -11.0 / 54.0, b52 = 2.5, b53 = -70.0 / 27.0, b54 = 35.0 / 27.0;
    static const double b61 = 1631.0 / 55296.0, b62 = 175.0 / 512.0, b63 = 575.0 / 13824.0, b64 = 44275.0 / 110592.0,
                        b65 = 253.0 / 4096.0;
    static const double c1 = 37.0 / 378.0, c3 = 250.0 / 621.0, c4 = 125.0 / 594.0, c6 = 512.0 / 1771.0;
    static const double d1 = c1 - 2825.0 / 27648.0, d3 = c3 - 18575.0 / 48384.0, d4 = c4 - 13525.0 / 55296.0,
                        d5 = -277.0 / 14336.0, d6 = c6 - 0.25;
    (void)a2;
    double k1[6], k2[6], k3[6], k4[6], k5[6], k6[6], t[6];
    rhs(p, y, k1);
    for (int i = 0; i < 6; ++i) t[i] = y[i] + h * (b21 * k1[i]);
    rhs(p, t, k2);
    for (int i = 0; i < 6; ++i) t[i] = y[i] + h * (b31 * k1[i] + b32 * k2[i]);
    rhs(p, t, k3);
    for (int i = 0; i < 6; ++i) t[i] = y[i] + h * (b41 * k1[i] + b42 * k2[i] + b43 * k3[i]);
    rhs(p, t, k4);
    for (int i = 0; i < 6; ++i) t[i] = y[i] + h * (b51 * k1[i] + b52 * k2[i] + b53 * k3[i] + b54 * k4[i]);
    rhs(p, t, k5);
    for (int i = 0; i < 6; ++i) t[i] = y[i] + h * (b61 * k1[i] + b62 * k2[i] + b63 * k3[i] + b64 * k4[i] + b65 * k5[i]);
    rhs(p, t, k6);
    for (int i = 0; i < 6; ++i) {
        y5[i] = y[i] + h * (c1 * k1[i] + c3 * k3[i] + c4 * k4[i] + c6 * k6[i]);
        err[i] = h * (d1 * k1[i] + d3 * k3[i] + d4 * k4[i] + d5 * k5[i] + d6 * k6[i]);
    }
}

// Advance one neuron over one time step of length h_step (C23, C24).  Returns true if it spiked.
inline bool step(const Params& p, State& s, double h_step) {
    double t = 0.0;
    bool spiked = false;
    while (t < h_step) {
        const double h = std::max(s.h_int, p.h_min);
        const bool clipped = h > h_step - t;                // the sub-step is cut short by the end of the time step
        const double h_try = clipped ? h_step - t : h;
        double y5[6], er[6];
        cash_karp(p, s.y, h_try, y5, er);
        double e = 0.0;
        for (int i = 0; i < 6; ++i) e = std::max(e, std::fabs(er[i]) / p.tol[i]);
        const bool accept = e <= 1.0 || h_try <= p.h_min;
        double fac = e > 0.0 ? 0.9 * std::pow(e, -0.2) : 5.0;
        fac = std::min(5.0, std::max(0.2, fac));
        // a clipped sub-step that succeeds says nothing about the size the dynamics allow: keep h_int then
        if (!clipped || !accept) s.h_int = std::min(h_step, h_try * fac);
        if (accept) {
            for (int i = 0; i < 6; ++i) s.y[i] = y5[i];
            t = clipped ? h_step : t + h_try;
            if (s.y[0] >= p.V_peak) {                       // C24
                s.y[0] = p.V_reset;
                s.y[1] += p.b;
                spiked = true;                              // a second crossing in the same step is not recorded (C20)
            }
        }
    }
    return spiked;
}

}  // namespace adex
