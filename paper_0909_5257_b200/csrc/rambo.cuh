// heget-b200, steps a1-a2: Philox4x32-10 uniforms -> massless RAMBO -> jet cuts, one event per thread.
//
// PAPER.md:184 has the GPU generate "momenta of initial and final partons using random numbers" that the paper drew on
// the CPU and copied over; here the counter-based generator runs in the kernel, so nothing is copied.
// Readings: A7, A7b (RAMBO parametrisation and its projection back onto momentum conservation), A9 (cuts in the partonic CM frame), A17 (Philox counter layout,
// u = (k + 0.5) 2^-32), A18 (deterministic re-draw with attempt = 0, 1, 2, ...; cap 2^16 -> weight 0).
#pragma once
#include "device/heget_rt.cuh"

namespace hg {

struct RamboArgs {
    double sqrt_s, pt_min, eta_max, dr_min, w0;
    unsigned long long seed, first_event, n_events;
    double* mom; double* weight; unsigned int* tries;
};

template <int NF>
__global__ void __launch_bounds__(128) k_rambo(const RamboArgs a) {
    const unsigned long long e = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= a.n_events) return;
    const unsigned long long ge = a.first_event + e;
    const double TWO_PI = 6.28318530717958647692, PI = 3.14159265358979323846;
    double p[NF][4];
    unsigned int attempt = 0; bool ok = false;
    for (; attempt < 65536u; ++attempt) {
        double q[NF][4], Q0 = 0, Q1 = 0, Q2 = 0, Q3 = 0;
#pragma unroll
        for (int i = 0; i < NF; ++i) {
            uint32_t r[4];
            philox4x32_10((uint32_t)ge, (uint32_t)(ge >> 32), attempt, (uint32_t)i, (uint32_t)a.seed, (uint32_t)(a.seed >> 32), r);
            const double u1 = ((double)r[0] + 0.5) * (1.0 / 4294967296.0), u2 = ((double)r[1] + 0.5) * (1.0 / 4294967296.0);
            const double u3 = ((double)r[2] + 0.5) * (1.0 / 4294967296.0), u4 = ((double)r[3] + 0.5) * (1.0 / 4294967296.0);
            const double c = 2.0 * u1 - 1.0, s = sqrt(1.0 - c * c), q0 = -log(u3 * u4);
            double sn, cs; sincos(TWO_PI * u2, &sn, &cs);
            q[i][0] = q0; q[i][1] = q0 * s * cs; q[i][2] = q0 * s * sn; q[i][3] = q0 * c;
            Q0 += q[i][0]; Q1 += q[i][1]; Q2 += q[i][2]; Q3 += q[i][3];
        }
        const double M = sqrt(Q0 * Q0 - Q1 * Q1 - Q2 * Q2 - Q3 * Q3);
        const double b0 = -Q1 / M, b1 = -Q2 / M, b2 = -Q3 / M, x = a.sqrt_s / M, gamma = Q0 / M, aa = 1.0 / (1.0 + gamma);
        double d1 = 0, d2 = 0, d3 = 0;
#pragma unroll
        for (int i = 0; i < NF; ++i) {
            const double bq = b0 * q[i][1] + b1 * q[i][2] + b2 * q[i][3];
            p[i][1] = x * (q[i][1] + b0 * q[i][0] + aa * bq * b0);
            p[i][2] = x * (q[i][2] + b1 * q[i][0] + aa * bq * b1);
            p[i][3] = x * (q[i][3] + b2 * q[i][0] + aa * bq * b2);
            d1 += p[i][1]; d2 += p[i][2]; d3 += p[i][3];
        }
        // reading A7b: back onto the constraint surface -- the boost loses eps*gamma^2 of momentum conservation
        double Et = 0;
#pragma unroll
        for (int i = 0; i < NF; ++i) {
            p[i][1] -= d1 / (double)NF; p[i][2] -= d2 / (double)NF; p[i][3] -= d3 / (double)NF;
            p[i][0] = sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2] + p[i][3] * p[i][3]);
            Et += p[i][0];
        }
        const double rs = a.sqrt_s / Et;
        ok = true;
        double eta[NF], phi[NF];
#pragma unroll
        for (int i = 0; i < NF; ++i) {
            p[i][0] *= rs; p[i][1] *= rs; p[i][2] *= rs; p[i][3] *= rs;
            const double pt2 = p[i][1] * p[i][1] + p[i][2] * p[i][2];
            const double pt = sqrt(pt2), pp = sqrt(pt2 + p[i][3] * p[i][3]);
            eta[i] = atanh(p[i][3] / pp);
            phi[i] = atan2(p[i][2], p[i][1]);
            if (a.pt_min > 0.0 && !(pt > a.pt_min)) ok = false;
            if (a.eta_max > 0.0 && !(fabs(eta[i]) < a.eta_max)) ok = false;
        }
        if (ok && a.dr_min > 0.0) {
#pragma unroll
            for (int i = 0; i < NF; ++i)
#pragma unroll
                for (int j = i + 1; j < NF; ++j) {
                    const double deta = eta[i] - eta[j];
                    double dphi = phi[i] - phi[j];
                    if (dphi > PI) dphi -= TWO_PI;
                    if (dphi <= -PI) dphi += TWO_PI;
                    if (!(sqrt(deta * deta + dphi * dphi) > a.dr_min)) ok = false;
                }
        }
        if (ok) break;
    }
    const size_t E = a.n_events;
    const double h = 0.5 * a.sqrt_s;
    a.mom[0 * E + e] = h; a.mom[1 * E + e] = 0.0; a.mom[2 * E + e] = 0.0; a.mom[3 * E + e] = h;
    a.mom[4 * E + e] = h; a.mom[5 * E + e] = 0.0; a.mom[6 * E + e] = 0.0; a.mom[7 * E + e] = -h;
#pragma unroll
    for (int i = 0; i < NF; ++i)
#pragma unroll
        for (int m = 0; m < 4; ++m) a.mom[((size_t)(2 + i) * 4 + m) * E + e] = p[i][m];
    if (a.weight) a.weight[e] = ok ? a.w0 : 0.0;
    if (a.tries) a.tries[e] = ok ? attempt + 1u : 65536u;
}

}  // namespace hg
