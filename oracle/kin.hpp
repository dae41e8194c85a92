// ORACLE (test infrastructure only).
//
// Textbook Feynman rules of massless QCD written out with explicit 4x4 Dirac matrices and
// explicit Lorentz-index loops -- deliberately slow and literal.  Nothing here follows the
// HELAS/HEGET "i-stripped" component formulas used on the GPU side.
//
// Lagrangian (signs as printed in the paper):
//   L_qqg  = - g T^a_{ij} A^a_mu  qbar_i gamma^mu q_j                     PAPER.md:226 (eq. 19)
//   L_ggg  = + g f^{abc} (d^mu A^{a nu}) A^b_mu A^c_nu                    PAPER.md:245 (eq. 23)
//   L_gggg = - g^2/4 f^{abe} f^{cde} A^{a mu} A^{b nu} A^c_mu A^d_nu      PAPER.md:319 (eq. 31)
// i.e. the usual QCD Lagrangian with covariant derivative d + i g T^a A^a.  The vertices
// derived from i*L (all momenta flowing INTO the vertex) are
//   qqg :  -i g gamma^mu T^a_{ij}
//   ggg :  -g f^{abc} [ g^{mu nu}(k1-k2)^rho + g^{nu rho}(k2-k3)^mu + g^{rho mu}(k3-k1)^nu ]
//   gggg:  -i g^2 [ f^{abe}f^{cde}(g^{mu rho}g^{nu sigma} - g^{mu sigma}g^{nu rho})
//                 + f^{ace}f^{bde}(g^{mu nu}g^{rho sigma} - g^{mu sigma}g^{nu rho})
//                 + f^{ade}f^{bce}(g^{mu nu}g^{rho sigma} - g^{mu rho}g^{nu sigma}) ]
// propagators: gluon (Feynman gauge)  -i g^{mu nu} delta^{ab} / k^2,
//              massless quark  i kslash delta_{ij} / k^2.
// Metric (+,-,-,-); momenta are (E, px, py, pz); Dirac matrices in the chiral representation
//   gamma^0 = [[0,1],[1,0]],  gamma^i = [[0,sigma^i],[-sigma^i,0]].
#pragma once
#include <complex>
#include <cmath>
#include "su3.hpp"

namespace orc {

static const double METRIC[4] = {1.0, -1.0, -1.0, -1.0};

struct Vec4 { cplx v[4]; };      // Lorentz vector, UPPER index
struct Spinor { cplx s[4]; };    // column spinor, or the entries of a row spinor

struct Gamma {
    cplx g[4][4][4];             // g[mu][row][col] = (gamma^mu)_{row col}
    Gamma() {
        const cplx I(0.0, 1.0);
        cplx sig[4][2][2];
        for (int m = 0; m < 4; ++m) for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) sig[m][i][j] = 0.0;
        sig[0][0][0] = 1.0; sig[0][1][1] = 1.0;
        sig[1][0][1] = 1.0; sig[1][1][0] = 1.0;
        sig[2][0][1] = -I;  sig[2][1][0] = I;
        sig[3][0][0] = 1.0; sig[3][1][1] = -1.0;
        for (int m = 0; m < 4; ++m) for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) g[m][i][j] = 0.0;
        for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) {
            g[0][i][2 + j] = sig[0][i][j];
            g[0][2 + i][j] = sig[0][i][j];
            for (int m = 1; m < 4; ++m) {
                g[m][i][2 + j] = sig[m][i][j];
                g[m][2 + i][j] = -sig[m][i][j];
            }
        }
    }
};
inline const Gamma& gam() { static Gamma G; return G; }

inline cplx mdot(const Vec4& a, const Vec4& b) {       // a^mu g_{mu nu} b^nu
    cplx r = 0.0;
    for (int m = 0; m < 4; ++m) r += METRIC[m] * a.v[m] * b.v[m];
    return r;
}
inline Vec4 real_vec(const double* p, double sign) {
    Vec4 r; for (int m = 0; m < 4; ++m) r.v[m] = sign * p[m]; return r;
}

// slash(k)_{row col} = k_mu gamma^mu = sum_mu METRIC[mu] k^mu gamma^mu
inline void slash(const Vec4& k, cplx out[4][4]) {
    const Gamma& G = gam();
    for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) {
        cplx r = 0.0;
        for (int m = 0; m < 4; ++m) r += METRIC[m] * k.v[m] * G.g[m][i][j];
        out[i][j] = r;
    }
}

// Massless helicity spinor u(p, h), h = +-1, with  pslash u = 0  and  gamma^5 u = h u
// (gamma^5 = diag(-1,-1,+1,+1) in this representation):
//   omega = sqrt(E + pz);  chi_+ = (omega, (px + i py)/omega);  chi_- = ((-px + i py)/omega, omega)
//   u_+ = (0, 0, chi_+),  u_- = (chi_-, 0, 0).        [SURVEY.md 8(c) oracle step 2]
// Along the -z axis (E + pz = 0, pT = 0) the limit is taken as chi_+ = (0, sqrt(2E)),
// chi_- = (-sqrt(2E), 0) (reading A19: any finite, normalised choice; phases are free, A14).
inline Spinor u_spinor(const double* p, int h) {
    Spinor u; for (int i = 0; i < 4; ++i) u.s[i] = 0.0;
    const double E = p[0], px = p[1], py = p[2], pz = p[3];
    const double pt2 = px * px + py * py;
    cplx chi0, chi1;
    if (pt2 == 0.0 && pz < 0.0) {
        const double w = std::sqrt(2.0 * E);
        if (h > 0) { chi0 = 0.0; chi1 = w; } else { chi0 = -w; chi1 = 0.0; }
    } else {
        const double w = std::sqrt(E + pz);
        if (h > 0) { chi0 = w; chi1 = cplx(px, py) / w; }
        else       { chi0 = cplx(-px, py) / w; chi1 = w; }
    }
    if (h > 0) { u.s[2] = chi0; u.s[3] = chi1; } else { u.s[0] = chi0; u.s[1] = chi1; }
    return u;
}
// Dirac conjugate  ubar = u^dagger gamma^0  (entries of the row spinor)
inline Spinor bar(const Spinor& u) {
    const Gamma& G = gam();
    Spinor r;
    for (int j = 0; j < 4; ++j) {
        cplx a = 0.0;
        for (int i = 0; i < 4; ++i) a += std::conj(u.s[i]) * G.g[0][i][j];
        r.s[j] = a;
    }
    return r;
}

// Polarisation vector of a massless vector boson with momentum p and helicity h = +-1:
//   eps1 = (0, px pz/(|p| pT), py pz/(|p| pT), -pT/|p|)   (theta-hat)
//   eps2 = (0, -py/pT, px/pT, 0)                          (phi-hat)
//   eps(h) = (-h eps1 - i eps2)/sqrt(2)                   [SURVEY.md 8(c) oracle step 2]
// pT = 0: eps1 = (0,1,0,0), eps2 = (0,0,sgn(pz),0) (A19).
// This is the wavefunction of an INCOMING boson; an outgoing one carries the complex conjugate.
inline Vec4 polvec(const double* p, int h) {
    const double px = p[1], py = p[2], pz = p[3];
    const double pt = std::sqrt(px * px + py * py);
    const double pp = std::sqrt(px * px + py * py + pz * pz);
    double e1[4], e2[4];
    e1[0] = 0.0; e2[0] = 0.0;
    if (pt == 0.0) {
        e1[1] = 1.0; e1[2] = 0.0; e1[3] = 0.0;
        e2[1] = 0.0; e2[2] = (pz >= 0.0) ? 1.0 : -1.0; e2[3] = 0.0;
    } else {
        e1[1] = px * pz / (pp * pt); e1[2] = py * pz / (pp * pt); e1[3] = -pt / pp;
        e2[1] = -py / pt;            e2[2] = px / pt;             e2[3] = 0.0;
    }
    const double r2 = 1.0 / std::sqrt(2.0);
    Vec4 e;
    for (int m = 0; m < 4; ++m) e.v[m] = cplx(-double(h) * e1[m] * r2, -e2[m] * r2);
    return e;
}
inline Vec4 conj(const Vec4& a) { Vec4 r; for (int m = 0; m < 4; ++m) r.v[m] = std::conj(a.v[m]); return r; }

// ---- vertices (colour stripped); all Lorentz vectors carry UPPER indices -----------------

// ggg: returns the amputated third leg  out^rho  (index raised) of
//   -g [ g_{mu nu}(k1-k2)_rho + g_{nu rho}(k2-k3)_mu + g_{rho mu}(k3-k1)_nu ] e1^mu e2^nu,
// momenta k1,k2,k3 all flowing into the vertex; colour factor f^{abc}, (a,b,c) <-> (1,2,3).
inline Vec4 vertex_ggg(double g, const Vec4& e1, const Vec4& k1, const Vec4& e2, const Vec4& k2, const Vec4& k3) {
    Vec4 out;
    for (int rho = 0; rho < 4; ++rho) {
        cplx acc = 0.0;
        for (int mu = 0; mu < 4; ++mu) for (int nu = 0; nu < 4; ++nu) {
            cplx V = 0.0;   // tensor with all indices LOWER
            if (mu == nu)  V += METRIC[mu] * METRIC[rho] * (k1.v[rho] - k2.v[rho]);
            if (nu == rho) V += METRIC[nu] * METRIC[mu] * (k2.v[mu] - k3.v[mu]);
            if (rho == mu) V += METRIC[rho] * METRIC[nu] * (k3.v[nu] - k1.v[nu]);
            acc += V * e1.v[mu] * e2.v[nu];
        }
        out.v[rho] = -g * acc * METRIC[rho];    // raise rho
    }
    return out;
}

// gggg, colour structure `piece` (legs a,b,c,d <-> e1,e2,e3,out; indices mu,nu,rho,sigma):
//   piece 0: f^{abe}f^{cde}: g_{mu rho}g_{nu sigma} - g_{mu sigma}g_{nu rho}
//   piece 1: f^{ace}f^{bde}: g_{mu nu}g_{rho sigma} - g_{mu sigma}g_{nu rho}
//   piece 2: f^{ade}f^{bce}: g_{mu nu}g_{rho sigma} - g_{mu rho}g_{nu sigma}
// times -i g^2; returns out^sigma (raised).
inline Vec4 vertex_gggg(double g, int piece, const Vec4& e1, const Vec4& e2, const Vec4& e3) {
    Vec4 out;
    for (int sg = 0; sg < 4; ++sg) {
        cplx acc = 0.0;
        for (int mu = 0; mu < 4; ++mu) for (int nu = 0; nu < 4; ++nu) for (int rho = 0; rho < 4; ++rho) {
            const double g_mn = (mu == nu) ? METRIC[mu] : 0.0, g_rs = (rho == sg) ? METRIC[rho] : 0.0;
            const double g_mr = (mu == rho) ? METRIC[mu] : 0.0, g_ns = (nu == sg) ? METRIC[nu] : 0.0;
            const double g_ms = (mu == sg) ? METRIC[mu] : 0.0, g_nr = (nu == rho) ? METRIC[nu] : 0.0;
            double W;
            if (piece == 0)      W = g_mr * g_ns - g_ms * g_nr;
            else if (piece == 1) W = g_mn * g_rs - g_ms * g_nr;
            else                 W = g_mn * g_rs - g_mr * g_ns;
            if (W != 0.0) acc += W * e1.v[mu] * e2.v[nu] * e3.v[rho];
        }
        out.v[sg] = cplx(0.0, -g * g) * acc * METRIC[sg];
    }
    return out;
}

// qqg, gluon leg open:  out^mu = psibar (-i g gamma^mu) psi ; colour T^a_{ij} (i: psibar, j: psi)
inline Vec4 vertex_qqg_gluon(double g, const Spinor& psibar, const Spinor& psi) {
    const Gamma& G = gam();
    Vec4 out;
    for (int mu = 0; mu < 4; ++mu) {
        cplx acc = 0.0;
        for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) acc += psibar.s[i] * G.g[mu][i][j] * psi.s[j];
        out.v[mu] = cplx(0.0, -g) * acc;
    }
    return out;
}
// qqg, outgoing-arrow leg open:  out = (-i g) epsslash psi   (column spinor)
inline Spinor vertex_qqg_psi(double g, const Vec4& eps, const Spinor& psi) {
    cplx E[4][4]; slash(eps, E);
    Spinor out;
    for (int i = 0; i < 4; ++i) {
        cplx acc = 0.0;
        for (int j = 0; j < 4; ++j) acc += E[i][j] * psi.s[j];
        out.s[i] = cplx(0.0, -g) * acc;
    }
    return out;
}
// qqg, incoming-arrow leg open:  out = psibar (-i g) epsslash   (row spinor)
inline Spinor vertex_qqg_psibar(double g, const Spinor& psibar, const Vec4& eps) {
    cplx E[4][4]; slash(eps, E);
    Spinor out;
    for (int j = 0; j < 4; ++j) {
        cplx acc = 0.0;
        for (int i = 0; i < 4; ++i) acc += psibar.s[i] * E[i][j];
        out.s[j] = cplx(0.0, -g) * acc;
    }
    return out;
}

// ---- propagators ------------------------------------------------------------------------
inline Vec4 prop_gluon(const Vec4& amp, const Vec4& k) {         // -i g^{mu nu}/k^2 . amp_nu
    const cplx k2 = mdot(k, k);
    Vec4 r; for (int m = 0; m < 4; ++m) r.v[m] = cplx(0.0, -1.0) * amp.v[m] / k2;
    return r;
}
inline Spinor prop_psi(const Spinor& amp, const Vec4& q) {       // (i qslash/q^2) amp ; q along the arrow
    cplx Q[4][4]; slash(q, Q);
    const cplx q2 = mdot(q, q);
    Spinor r;
    for (int i = 0; i < 4; ++i) {
        cplx acc = 0.0;
        for (int j = 0; j < 4; ++j) acc += Q[i][j] * amp.s[j];
        r.s[i] = cplx(0.0, 1.0) * acc / q2;
    }
    return r;
}
inline Spinor prop_psibar(const Spinor& amp, const Vec4& q) {    // amp (i qslash/q^2) ; q along the arrow
    cplx Q[4][4]; slash(q, Q);
    const cplx q2 = mdot(q, q);
    Spinor r;
    for (int j = 0; j < 4; ++j) {
        cplx acc = 0.0;
        for (int i = 0; i < 4; ++i) acc += amp.s[i] * Q[i][j];
        r.s[j] = cplx(0.0, 1.0) * acc / q2;
    }
    return r;
}
}  // namespace orc
