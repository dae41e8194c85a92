// ORACLE (test infrastructure only).
//
// Evaluation of eq. 4 for one phase-space point, the literal way:
//   me2 = S * 1/4 * 1/(n_a n_b) * sum_{helicities} sum_{colours} | sum_{diagrams l} (M_lambda)_l^{c} |^2
// Tier O2 (paper's method, eqs. 8-10):  J_alpha = sum_l coef_{alpha l} A_l,
//   sum_c |M^c|^2 = sum_{alpha beta} J_alpha C_{alpha beta} J_beta^*.
// Tier O1 (no colour basis at all):  sum_c | sum_l D_l^c A_l |^2 over every colour assignment c.
// A_l is the colour-stripped kinematic factor of diagram l (for a gggg vertex: of one of its three
// colour structures), built from kin.hpp's vertices and propagators along the tree.
#pragma once
#include "kin.hpp"
#include "diagrams.hpp"
#include "colour.hpp"

namespace orc {

struct Model {
    DiagramSet D;
    ColourData cd;
    double gs;            // g_s = sqrt(4 pi alpha_s)
};

struct NodeValue { Vec4 vec; Spinor sp; };   // "propagated" value handed to the parent

// mom: physical momenta p[leg][4]; hel[leg] = +-1 physical helicities; ward_leg >= 0 replaces that gluon's
// polarisation vector by its momentum (gauge-invariance check).  Fills A[l] for every diagram l.
inline void diagram_amplitudes(const Model& M, const double (*p)[4], const int* hel, int ward_leg, std::vector<cplx>& A) {
    const DiagramSet& D = M.D;
    const Process& P = D.proc;
    const int n = P.n_ext();
    const double g = M.gs;
    // momenta flowing INTO the diagram
    Vec4 k[16];
    for (int i = 0; i < n; ++i) k[i] = real_vec(p[i], P.legs[i].initial ? +1.0 : -1.0);
    // external wavefunctions
    Vec4 wv[16]; Spinor ws[16];
    for (int i = 0; i < n; ++i) {
        const Leg& L = P.legs[i];
        if (L.kind == LEG_G) {
            Vec4 e = polvec(p[i], hel[i]);
            wv[i] = L.initial ? e : conj(e);
            if (i == ward_leg) wv[i] = real_vec(p[i], 1.0);
        } else if (L.kind == LEG_IN) {
            // initial quark u(p,h); final antiquark v(p,h) = u(p,-h) (massless, phase free: A14)
            ws[i] = L.initial ? u_spinor(p[i], hel[i]) : u_spinor(p[i], -hel[i]);
        } else {
            // final quark ubar(p,h); initial antiquark vbar(p,h) = ubar(p,-h)
            ws[i] = L.initial ? bar(u_spinor(p[i], -hel[i])) : bar(u_spinor(p[i], hel[i]));
        }
    }
    const size_t nn = D.nodes.size();
    std::vector<NodeValue> amp(nn), prop(nn);     // amputated / with propagator
    std::vector<Vec4> kS(nn);
    for (size_t id = 0; id < nn; ++id) {
        const Node& nd = D.nodes[id];
        Vec4 ks; for (int m = 0; m < 4; ++m) ks.v[m] = 0.0;
        for (int i = 0; i < n; ++i) if ((nd.mask >> i) & 1u) for (int m = 0; m < 4; ++m) ks.v[m] += k[i].v[m];
        kS[id] = ks;
        if (nd.kind == NK_LEAF) {
            if (nd.ptype == PT_G) { amp[id].vec = wv[nd.leg]; prop[id].vec = wv[nd.leg]; }
            else { amp[id].sp = ws[nd.leg]; prop[id].sp = ws[nd.leg]; }
            continue;
        }
        const int c0 = nd.ch[0], c1 = nd.ch[1], c2 = nd.ch[2];
        Vec4 mks; for (int m = 0; m < 4; ++m) mks.v[m] = -ks.v[m];
        switch (nd.kind) {
        case NK_GGG:
            amp[id].vec = vertex_ggg(g, prop[c0].vec, kS[c0], prop[c1].vec, kS[c1], mks);
            prop[id].vec = prop_gluon(amp[id].vec, ks);
            break;
        case NK_GGGG:
            amp[id].vec = vertex_gggg(g, nd.piece, prop[c0].vec, prop[c1].vec, prop[c2].vec);
            prop[id].vec = prop_gluon(amp[id].vec, ks);
            break;
        case NK_QQG_G:
            amp[id].vec = vertex_qqg_gluon(g, prop[c0].sp, prop[c1].sp);
            prop[id].vec = prop_gluon(amp[id].vec, ks);
            break;
        case NK_QG_Q:      // momentum along the arrow = momentum flowing from the leaves to the root
            amp[id].sp = vertex_qqg_psi(g, prop[c1].vec, prop[c0].sp);
            prop[id].sp = prop_psi(amp[id].sp, ks);
            break;
        case NK_BG_B:      // arrow runs from the root to the leaves: momentum along it is -k_S
            amp[id].sp = vertex_qqg_psibar(g, prop[c0].sp, prop[c1].vec);
            prop[id].sp = prop_psibar(amp[id].sp, mks);
            break;
        default: break;
        }
    }
    const int r = D.root;
    A.resize(D.diagrams.size());
    for (size_t l = 0; l < D.diagrams.size(); ++l) {
        const int id = D.diagrams[l];
        cplx a = 0.0;
        if (P.legs[r].kind == LEG_G) a = mdot(wv[r], amp[id].vec);
        else for (int i = 0; i < 4; ++i) a += ws[r].s[i] * amp[id].sp.s[i];   // row . column either way
        A[l] = a * (double)D.diagram_sign[l];
    }
}

inline void colour_amplitudes(const Model& M, const std::vector<cplx>& A, std::vector<cplx>& J) {
    J.assign(M.cd.m, 0.0);
    for (size_t l = 0; l < A.size(); ++l)
        for (size_t t = 0; t < M.cd.coef[l].size(); ++t) J[M.cd.coef[l][t].first] += M.cd.coef[l][t].second * A[l];
}

inline double colour_sum_O2(const Model& M, const std::vector<cplx>& J) {       // eq. 10
    const int m = M.cd.m;
    double s = 0.0;
    for (int a = 0; a < m; ++a) for (int b = 0; b < m; ++b) s += (J[a] * M.cd.C[(size_t)a * m + b] * std::conj(J[b])).real();
    return s;
}

inline double colour_sum_O1(const Model& M, const std::vector<cplx>& A) {       // eq. 4 + eq. 7, colour by colour
    std::vector<cplx> Mc(M.cd.n_assign, 0.0);
    for (size_t l = 0; l < A.size(); ++l) {
        const SparseVec& d = M.cd.diag_colour[l];
        for (size_t k = 0; k < d.idx.size(); ++k) Mc[d.idx[k]] += d.val[k] * A[l];
    }
    double s = 0.0;
    for (size_t c = 0; c < Mc.size(); ++c) s += std::norm(Mc[c]);
    return s;
}

// helicity- and colour-summed, averaged |M|^2 of one event; tier = 1 or 2
inline double me2_event(const Model& M, const double (*p)[4], int tier) {
    const Process& P = M.D.proc;
    const int n = P.n_ext();
    std::vector<cplx> A, J;
    double sum = 0.0;
    int hel[16];
    for (int h = 0; h < (1 << n); ++h) {
        for (int i = 0; i < n; ++i) hel[i] = ((h >> i) & 1) ? +1 : -1;
        diagram_amplitudes(M, p, hel, -1, A);
        if (tier == 1) sum += colour_sum_O1(M, A);
        else { colour_amplitudes(M, A, J); sum += colour_sum_O2(M, J); }
    }
    return sum * P.sym_factor * P.avg_spin * P.avg_color;
}
}  // namespace orc
