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
#include "kin.hpp"

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
}  // namespace orc
