// ORACLE (test infrastructure only).
//
// Steps a1-a2 of the hot path: Philox4x32-10 counter-based uniforms, massless
// RAMBO phase-space points in the partonic centre-of-mass frame, and the jet cuts.
//
// PAPER.md:184 ("generation of ... momenta of initial and final partons using random numbers")
// gives no parametrisation; BASELINE.json fixes massless RAMBO with a Philox counter-based
// generator.  Readings taken:
//  A7  per final particle i one Philox block -> uniforms u1..u4:
//        c = 2 u1 - 1, phi = 2 pi u2, q0 = -ln(u3 u4), q = q0 (1, s cos phi, s sin phi, c), s = sqrt(1-c^2)
//      Q = sum q, M = sqrt(Q^2), b = -Q_vec/M, x = sqrt(s_hat)/M, gamma = Q0/M, a = 1/(1+gamma)
//        p0 = x (gamma q0 + b.q),  p_vec = x (q_vec + b q0 + a (b.q) b)
//      weight w0 = (pi/2)^(n-1) s_hat^(n-2) / ((n-1)! (n-2)!) (2 pi)^(4-3n)
//  A7b after the boost the point is put back on the constraint surface (see rambo_attempt): floating-point RAMBO
//      misses momentum conservation by eps Q0^2/M^2, which reaches 1e-10 among 10^4 two-body events
//  A17 Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): multipliers 0xD2511F53, 0xCD9E8D57, Weyl key
//      increments 0x9E3779B9, 0xBB67AE85, 10 rounds; counter = (event_lo, event_hi, attempt, particle),
//      key = (seed_lo, seed_hi); uniform u = (k + 0.5) 2^-32.
//  A9  cuts in the partonic CM frame: pT > pt_min, |eta| < eta_max, Delta R_ij > dr_min (strict),
//      eta = atanh(pz/|p|), Delta phi wrapped to (-pi, pi]; cf. PAPER.md:118-135 (eqs. 14, 15b).
//  A18 events failing the cuts are re-drawn with attempt = 0,1,2,... (cap 2^16 -> weight 0).
#pragma once
#include <cstdint>
#include <cmath>

namespace orc {

inline void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        const uint64_t m0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        const uint64_t m1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(m0 >> 32), lo0 = (uint32_t)m0;
        const uint32_t hi1 = (uint32_t)(m1 >> 32), lo1 = (uint32_t)m1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

inline double u01(uint32_t k) { return ((double)k + 0.5) * (1.0 / 4294967296.0); }

struct Cuts { double pt_min, eta_max, dr_min; };   // <= 0 disables a cut

// final-state momenta p[n][4] = (E,px,py,pz); returns true if all cuts pass
inline bool pass_cuts(int n, const double (*p)[4], const Cuts& cuts) {
    const double PI = 3.14159265358979323846;
    double eta[16], phi[16];
    for (int i = 0; i < n; ++i) {
        const double pt = std::sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2]);
        const double pp = std::sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2] + p[i][3] * p[i][3]);
        eta[i] = std::atanh(p[i][3] / pp);
        phi[i] = std::atan2(p[i][2], p[i][1]);
        if (cuts.pt_min > 0.0 && !(pt > cuts.pt_min)) return false;
        if (cuts.eta_max > 0.0 && !(std::fabs(eta[i]) < cuts.eta_max)) return false;
    }
    if (cuts.dr_min > 0.0)
        for (int i = 0; i < n; ++i) for (int j = i + 1; j < n; ++j) {
            const double deta = eta[i] - eta[j];
            double dphi = phi[i] - phi[j];
            if (dphi > PI) dphi -= 2.0 * PI;
            if (dphi <= -PI) dphi += 2.0 * PI;
            const double dr = std::sqrt(deta * deta + dphi * dphi);
            if (!(dr > cuts.dr_min)) return false;
        }
    return true;
}

// One RAMBO attempt.  n = number of final-state particles (2..14).
inline void rambo_attempt(int n, double sqrt_s, uint64_t seed, uint64_t event, uint32_t attempt, double (*p)[4]) {
    const double PI = 3.14159265358979323846;
    double q[16][4];
    double Q[4] = {0, 0, 0, 0};
    const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
    for (int i = 0; i < n; ++i) {
        const uint32_t ctr[4] = {(uint32_t)(event & 0xffffffffu), (uint32_t)(event >> 32), attempt, (uint32_t)i};
        uint32_t r[4];
        philox4x32_10(ctr, key, r);
        const double u1 = u01(r[0]), u2 = u01(r[1]), u3 = u01(r[2]), u4 = u01(r[3]);
        const double c = 2.0 * u1 - 1.0;
        const double s = std::sqrt(1.0 - c * c);
        const double ph = 2.0 * PI * u2;
        const double q0 = -std::log(u3 * u4);
        q[i][0] = q0; q[i][1] = q0 * s * std::cos(ph); q[i][2] = q0 * s * std::sin(ph); q[i][3] = q0 * c;
        for (int m = 0; m < 4; ++m) Q[m] += q[i][m];
    }
    const double M = std::sqrt(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
    const double b[3] = {-Q[1] / M, -Q[2] / M, -Q[3] / M};
    const double x = sqrt_s / M;
    const double gamma = Q[0] / M;
    const double a = 1.0 / (1.0 + gamma);
    for (int i = 0; i < n; ++i) {
        const double bq = b[0] * q[i][1] + b[1] * q[i][2] + b[2] * q[i][3];
        p[i][0] = x * (gamma * q[i][0] + bq);
        for (int k = 0; k < 3; ++k) p[i][1 + k] = x * (q[i][1 + k] + b[k] * q[i][0] + a * bq * b[k]);
    }
    // A7b: the boost above forms each p_i from terms gamma^2 times larger than the result (gamma = Q0/M), so in
    // floating point sum p_i misses (sqrt_s, 0, 0, 0) by ~ eps gamma^2 sqrt_s, and gamma^2 has a 1/G tail for n = 2.
    // The point is put back on the constraint surface: remove the residual 3-momentum evenly, set E_i = |p_i|
    // (exactly massless), rescale to sum E_i = sqrt_s.  The shift is of the size of the rounding error it removes.
    double d[3] = {0, 0, 0};
    for (int i = 0; i < n; ++i) for (int k = 0; k < 3; ++k) d[k] += p[i][1 + k];
    double Et = 0;
    for (int i = 0; i < n; ++i) {
        for (int k = 0; k < 3; ++k) p[i][1 + k] -= d[k] / (double)n;
        p[i][0] = std::sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2] + p[i][3] * p[i][3]);
        Et += p[i][0];
    }
    const double r = sqrt_s / Et;
    for (int i = 0; i < n; ++i) for (int m = 0; m < 4; ++m) p[i][m] *= r;
}

inline double rambo_flat_weight(int n, double sqrt_s) {
    const double PI = 3.14159265358979323846;
    double w = std::pow(PI / 2.0, n - 1) * std::pow(sqrt_s * sqrt_s, n - 2) * std::pow(2.0 * PI, 4 - 3 * n);
    for (int k = 2; k <= n - 1; ++k) w /= (double)k;
    for (int k = 2; k <= n - 2; ++k) w /= (double)k;
    return w;
}

// Fills SoA momenta mom[(leg*4+mu)*n_events + e] for legs 0,1 (beams) and 2..n+1 (finals).
inline void sample_momenta(int n_final, double sqrt_s, const Cuts& cuts, uint64_t seed, uint64_t first_event,
                           uint64_t n_events, double* mom, double* weight, uint32_t* tries) {
    const double w0 = rambo_flat_weight(n_final, sqrt_s);
    #pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < (int64_t)n_events; ++e) {
        double p[16][4];
        uint32_t attempt = 0;
        bool ok = false;
        for (; attempt < 65536u; ++attempt) {
            rambo_attempt(n_final, sqrt_s, seed, first_event + (uint64_t)e, attempt, p);
            if (pass_cuts(n_final, p, cuts)) { ok = true; break; }
        }
        const double h = 0.5 * sqrt_s;
        const double beam[2][4] = {{h, 0.0, 0.0, h}, {h, 0.0, 0.0, -h}};
        for (int m = 0; m < 4; ++m) {
            mom[(0 * 4 + m) * n_events + e] = beam[0][m];
            mom[(1 * 4 + m) * n_events + e] = beam[1][m];
            for (int i = 0; i < n_final; ++i) mom[((2 + i) * 4 + m) * n_events + e] = p[i][m];
        }
        if (weight) weight[e] = ok ? w0 : 0.0;
        if (tries) tries[e] = ok ? attempt + 1 : 65536u;
    }
}
}  // namespace orc
