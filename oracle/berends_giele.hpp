// ORACLE (test infrastructure only) -- tier O3: colour-ordered Berends-Giele
// recursion for n-gluon partial amplitudes.  It knows nothing about diagrams.hpp / colour.hpp: no
// diagram list, no colour tensors.  It is used only to cross-check the diagram-built J_alpha.
//
// Colour-ordered rules derived from kin.hpp's full rules with f^{abc} = -2i Tr([T^a,T^b]T^c) and
// sum_a Tr(X T^a) Tr(T^a Y) = Tr(XY)/2 - Tr(X)Tr(Y)/6 (the 1/6 terms cancel between gluons):
//   3-vertex for cyclic order (1,2,3):  2 i g [ g_{mu nu}(k1-k2)_rho + g_{nu rho}(k2-k3)_mu + g_{rho mu}(k3-k1)_nu ]
//   4-vertex for cyclic order (1,2,3,4): 2 i g^2 [ 2 g_{mu rho} g_{nu sigma} - g_{mu nu} g_{rho sigma} - g_{mu sigma} g_{nu rho} ]
//   propagator: (1/2) (-i g^{mu nu}) / K^2
// so that the full amplitude is  sum_sigma Tr(T^{a_s(0)} ... T^{a_s(n-1)}) * A(s(0),...,s(n-1))  over
// non-cyclic orderings -- the expansion of eq. 8 / eq. 17.
#pragma once
#include <algorithm>
#include <vector>
#include "kin.hpp"
#include "su3.hpp"

namespace orc {

inline Vec4 bg_v3(const Vec4& J1, const Vec4& k1, const Vec4& J2, const Vec4& k2) {
    Vec4 a, b, out;
    for (int m = 0; m < 4; ++m) { a.v[m] = k1.v[m] + 2.0 * k2.v[m]; b.v[m] = 2.0 * k1.v[m] + k2.v[m]; }
    const cplx j12 = mdot(J1, J2), aJ1 = mdot(a, J1), bJ2 = mdot(b, J2);
    for (int m = 0; m < 4; ++m) out.v[m] = j12 * (k1.v[m] - k2.v[m]) + aJ1 * J2.v[m] - bJ2 * J1.v[m];
    return out;
}
inline Vec4 bg_v4(const Vec4& J1, const Vec4& J2, const Vec4& J3) {
    const cplx j13 = mdot(J1, J3), j12 = mdot(J1, J2), j23 = mdot(J2, J3);
    Vec4 out;
    for (int m = 0; m < 4; ++m) out.v[m] = 2.0 * j13 * J2.v[m] - j12 * J3.v[m] - j23 * J1.v[m];
    return out;
}

// physical momenta p[leg][4], physical helicities hel[leg], legs 0,1 incoming; order[n] = trace order
inline cplx bg_partial_amplitude(int n, const double (*p)[4], const int* hel, const int* order, double g) {
    Vec4 k[16], eps[16];
    for (int i = 0; i < n; ++i) {
        const int leg = order[i];
        const bool initial = leg < 2;
        k[i] = real_vec(p[leg], initial ? +1.0 : -1.0);
        Vec4 e = polvec(p[leg], hel[leg]);
        eps[i] = initial ? e : conj(e);
    }
    // J[i][j]: current of ordered legs i..j (inclusive), i<=j<=n-2, propagator included for j>i
    static thread_local Vec4 J[16][16], K[16][16], V[16][16];
    for (int i = 0; i < n - 1; ++i) { J[i][i] = eps[i]; K[i][i] = k[i]; }
    for (int len = 2; len <= n - 1; ++len)
        for (int i = 0; i + len - 1 <= n - 2; ++i) {
            const int j = i + len - 1;
            Vec4 acc; for (int m = 0; m < 4; ++m) acc.v[m] = 0.0;
            for (int m = 0; m < 4; ++m) K[i][j].v[m] = K[i][j - 1].v[m] + k[j].v[m];
            for (int s = i; s < j; ++s) {
                Vec4 t = bg_v3(J[i][s], K[i][s], J[s + 1][j], K[s + 1][j]);
                for (int m = 0; m < 4; ++m) acc.v[m] += cplx(0.0, 2.0 * g) * t.v[m];
            }
            for (int s = i; s < j; ++s) for (int t2 = s + 1; t2 < j; ++t2) {
                Vec4 t = bg_v4(J[i][s], J[s + 1][t2], J[t2 + 1][j]);
                for (int m = 0; m < 4; ++m) acc.v[m] += cplx(0.0, 2.0 * g * g) * t.v[m];
            }
            V[i][j] = acc;                                           // amputated
            const cplx K2 = mdot(K[i][j], K[i][j]);
            for (int m = 0; m < 4; ++m) J[i][j].v[m] = cplx(0.0, -0.5) * acc.v[m] / K2;
        }
    return mdot(eps[n - 1], V[0][n - 2]);
}

// Tier O1 colour definition on tier O3 kinematics, for pure-gluon processes too large for diagrams.hpp / colour.hpp (g g -> 5 g:
// 7245 diagrams, 720 traces): the colour-summed squared amplitude of ONE helicity configuration,
//     sum over all 8^n colour assignments {c_i} of | sum_sigma Tr(T^{c_s(0)} ... T^{c_s(n-1)}) A(s(0), ..., s(n-1)) |^2
// (eq. 8 with the single-trace basis of eq. 17), sigma over the (n-1)! non-cyclic orderings with leg 0 first,
// A from the recursion above, the traces multiplied out with the numeric Gell-Mann matrices.  The orderings are walked in
// lexicographic order and the products T^{c_0} T^{c_s(1)} ... are kept as a stack of prefixes, so a step to the next ordering
// re-multiplies only the tail that changed (plain arithmetic, nothing skipped).
inline double gluon_colour_sum_bg(int n, const double (*p)[4], const int* hel, double g) {
    std::vector<int> rest(n - 1); for (int i = 0; i < n - 1; ++i) rest[i] = i + 1;
    std::vector<std::vector<int> > orders; std::vector<cplx> amp;
    do {
        std::vector<int> o(n); o[0] = 0; for (int i = 0; i < n - 1; ++i) o[i + 1] = rest[i];
        orders.push_back(o); amp.push_back(bg_partial_amplitude(n, p, hel, o.data(), g));
    } while (std::next_permutation(rest.begin(), rest.end()));
    const SU3& S = su3();
    long total = 1; for (int i = 0; i < n; ++i) total *= 8;
    double sum = 0.0;
    #pragma omp parallel for schedule(static) reduction(+ : sum)
    for (long code = 0; code < total; ++code) {
        int c[16]; long q = code; for (int i = 0; i < n; ++i) { c[i] = (int)(q % 8); q /= 8; }
        cplx pre[16][3][3];                       // pre[d] = T^{c_0} T^{c_o(1)} ... T^{c_o(d)}
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) pre[0][i][j] = S.T[c[0]][i][j];
        cplx M = 0.0;
        for (size_t s = 0; s < orders.size(); ++s) {
            int d0 = 1;
            if (s > 0) while (orders[s][d0] == orders[s - 1][d0]) ++d0;
            for (int d = d0; d < n; ++d) {
                const cplx (*T)[3] = S.T[c[orders[s][d]]];
                for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
                    cplx v = 0.0; for (int k = 0; k < 3; ++k) v += pre[d - 1][i][k] * T[k][j];
                    pre[d][i][j] = v;
                }
            }
            M += (pre[n - 1][0][0] + pre[n - 1][1][1] + pre[n - 1][2][2]) * amp[s];
        }
        sum += std::norm(M);
    }
    return sum;
}
}  // namespace orc
