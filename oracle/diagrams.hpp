// ORACLE (test infrastructure only).
//
// Process description and literal enumeration of every tree-level Feynman diagram of a
// massless-QCD process (eq. 7: "the summation is over all the Feynman diagrams").
//
// A diagram is a tree whose internal nodes are qqg, ggg or gggg vertices.  It is enumerated as a
// tree ROOTED at the last external leg: the other legs are grouped recursively into off-shell
// lines.  Children of a ggg / gggg vertex are unordered, so every split is generated once
// (the part holding the lowest leg first).  Following the paper's counting convention (reading
// A11, Table 1) a gggg vertex is entered three times, once per colour structure
// of eq. 36 -- `n_diagrams` counts those, `n_topologies` counts each once.
//
// Quark lines: every quark leg is the IN-end (fermion arrow enters the diagram: initial q,
// final qbar) or the OUT-end (initial qbar, final q) of a line.  For identical flavours every
// pairing of in-ends with out-ends is a separate set of diagrams with relative sign = parity of
// the pairing permutation (Fermi statistics; SURVEY.md 8(c) oracle step 4).
#pragma once
#include <vector>
#include <string>
#include <sstream>
#include <map>
#include <algorithm>
#include <stdexcept>

namespace orc {

enum LegKind { LEG_G = 0, LEG_IN = 1, LEG_OUT = 2 };      // gluon, quark-line in-end, out-end
struct Leg { int kind; int flavour; bool initial; bool anti; };

struct Process {
    std::vector<Leg> legs;          // legs[0], legs[1] initial, rest final, in process-string order
    int n_ext() const { return (int)legs.size(); }
    double sym_factor;              // 1 / prod k!  over identical final-state particles
    double avg_color;               // 1/(n_a n_b), n = 3 (q, qbar) or 8 (g)
    double avg_spin;                // 1/(2*2)
};

inline Process parse_process(const std::string& text) {
    Process P;
    std::istringstream in(text);
    std::string tok;
    bool final_state = false;
    while (in >> tok) {
        if (tok == ">" || tok == "->") { final_state = true; continue; }
        Leg L; L.initial = !final_state; L.anti = false; L.flavour = -1;
        if (tok == "g") { L.kind = LEG_G; }
        else {
            std::string f = tok;
            if (!f.empty() && f[f.size() - 1] == '~') { L.anti = true; f = f.substr(0, f.size() - 1); }
            const std::string names = "udsc";
            if (f.size() != 1 || names.find(f) == std::string::npos) throw std::runtime_error("unknown particle " + tok);
            L.flavour = (int)names.find(f);
            // arrow enters the diagram at an initial quark or a final antiquark
            L.kind = (L.initial != L.anti) ? LEG_IN : LEG_OUT;
        }
        P.legs.push_back(L);
    }
    int n_init = 0; for (size_t i = 0; i < P.legs.size(); ++i) n_init += P.legs[i].initial;
    if (n_init != 2 || P.legs.size() < 4 || P.legs.size() > 8) throw std::runtime_error("need 2 -> n, 2 <= n <= 6");
    // identical-particle factor: the final state is symmetrised over particles that cannot be told apart, i.e.
    // final legs with the same species (gluon / flavour) AND the same particle-antiparticle nature.  Counted pairwise from the
    // leg list: every final leg that has m identical final legs BEFORE it contributes 1/(m+1); the product is 1/prod k!.
    P.sym_factor = 1.0;
    for (size_t i = 2; i < P.legs.size(); ++i) {
        int earlier_twins = 0;
        for (size_t j = 2; j < i; ++j) {
            const Leg& a = P.legs[i]; const Leg& b = P.legs[j];
            const bool both_gluons = a.kind == LEG_G && b.kind == LEG_G;
            const bool same_quark = a.kind != LEG_G && b.kind != LEG_G && a.flavour == b.flavour && a.anti == b.anti;
            if (both_gluons || same_quark) ++earlier_twins;
        }
        P.sym_factor /= (double)(earlier_twins + 1);
    }
    const double na = (P.legs[0].kind == LEG_G) ? 8.0 : 3.0, nb = (P.legs[1].kind == LEG_G) ? 8.0 : 3.0;
    P.avg_color = 1.0 / (na * nb);
    P.avg_spin = 0.25;
    return P;
}

// A pairing = assignment of every in-end to an out-end of the same flavour.
struct Pairing {
    std::vector<int> line_of_leg;   // -1 for gluons
    std::vector<int> in_leg, out_leg;   // per line
    int sign;
};

inline std::vector<Pairing> enumerate_pairings(const Process& P) {
    std::vector<int> ins, outs;
    for (int i = 0; i < P.n_ext(); ++i) {
        if (P.legs[i].kind == LEG_IN) ins.push_back(i);
        if (P.legs[i].kind == LEG_OUT) outs.push_back(i);
    }
    if (ins.size() != outs.size()) throw std::runtime_error("quark number not conserved");
    std::vector<Pairing> result;
    std::vector<int> perm(outs.size());
    for (size_t i = 0; i < perm.size(); ++i) perm[i] = (int)i;
    do {
        bool ok = true;
        for (size_t i = 0; i < ins.size(); ++i)
            if (P.legs[ins[i]].flavour != P.legs[outs[perm[i]]].flavour) ok = false;
        if (!ok) continue;
        Pairing pr;
        pr.line_of_leg.assign(P.n_ext(), -1);
        for (size_t i = 0; i < ins.size(); ++i) {
            pr.in_leg.push_back(ins[i]); pr.out_leg.push_back(outs[perm[i]]);
            pr.line_of_leg[ins[i]] = (int)i; pr.line_of_leg[outs[perm[i]]] = (int)i;
        }
        int inv = 0;
        for (size_t i = 0; i < perm.size(); ++i) for (size_t j = i + 1; j < perm.size(); ++j) inv += perm[i] > perm[j];
        pr.sign = (inv % 2) ? -1 : +1;
        result.push_back(pr);
    } while (std::next_permutation(perm.begin(), perm.end()));
    if (result.empty()) throw std::runtime_error("flavour not conserved");
    // Fermi sign is relative: normalise so that the first pairing has sign +1
    const int s0 = result[0].sign;
    for (size_t i = 0; i < result.size(); ++i) result[i].sign *= s0;
    return result;
}

enum PType { PT_G = 0, PT_Q = 1, PT_B = 2, PT_NONE = 3 };   // gluon, psi (holds an in-end), psibar (holds an out-end)
enum NKind { NK_LEAF = 0, NK_GGG, NK_GGGG, NK_QQG_G, NK_QG_Q, NK_BG_B };

struct Node {
    int ptype, line;        // what flows out of this subtree towards the root
    unsigned mask;          // external legs contained
    int kind;
    int ch[3];              // children (node ids); NK_QQG_G: (psibar, psi); NK_QG_Q: (psi, g); NK_BG_B: (psibar, g)
    int piece;              // NK_GGGG: colour structure 0,1,2
    int leg;                // NK_LEAF
    int pairing;
    double n_topo_weight;   // 3^-(number of gggg vertices in the subtree): sums to the topology count
};

struct DiagramSet {
    Process proc;
    std::vector<Pairing> pairings;
    std::vector<Node> nodes;            // children always precede parents
    std::vector<int> diagrams;          // node ids over (all legs but the root) that close on the root
    std::vector<int> diagram_sign;      // Fermi sign of the pairing
    int root;                           // root leg = last leg
    double n_topologies;
};

class Enumerator {
public:
    Enumerator(DiagramSet& ds, int pairing) : D(ds), pr(ds.pairings[pairing]), ip(pairing) {}

    void classify(unsigned S, int& ptype, int& line) const {
        ptype = PT_G; line = -1;
        for (size_t l = 0; l < pr.in_leg.size(); ++l) {
            const bool hi = (S >> pr.in_leg[l]) & 1u, ho = (S >> pr.out_leg[l]) & 1u;
            if (hi == ho) continue;
            if (ptype != PT_G) { ptype = PT_NONE; return; }      // two open lines: no such particle
            ptype = hi ? PT_Q : PT_B; line = (int)l;
        }
    }

    const std::vector<int>& currents(unsigned S) {
        std::map<unsigned, std::vector<int> >::iterator it = memo.find(S);
        if (it != memo.end()) return it->second;
        std::vector<int> out;
        int ptype, line; classify(S, ptype, line);
        if ((S & (S - 1)) == 0) {                                 // single leg
            int leg = 0; while (!((S >> leg) & 1u)) ++leg;
            Node n; n.ptype = ptype; n.line = line; n.mask = S; n.kind = NK_LEAF; n.leg = leg; n.piece = 0;
            n.ch[0] = n.ch[1] = n.ch[2] = -1; n.pairing = ip; n.n_topo_weight = 1.0;
            out.push_back(add(n));
        } else if (ptype != PT_NONE) {
            const unsigned low = S & (~S + 1u);
            // two-way splits S = A + B, A holds the lowest leg
            for (unsigned A = (S - 1) & S; A; A = (A - 1) & S) {
                if (!(A & low)) continue;
                const unsigned B = S & ~A;
                int ta, la, tb, lb; classify(A, ta, la); classify(B, tb, lb);
                if (ta == PT_NONE || tb == PT_NONE) continue;
                const std::vector<int> ca = currents(A), cb = currents(B);
                for (size_t i = 0; i < ca.size(); ++i) for (size_t j = 0; j < cb.size(); ++j) {
                    Node n; n.ptype = ptype; n.line = line; n.mask = S; n.piece = 0; n.leg = -1; n.pairing = ip;
                    n.ch[2] = -1;
                    n.n_topo_weight = D.nodes[ca[i]].n_topo_weight * D.nodes[cb[j]].n_topo_weight;
                    if (ptype == PT_G && ta == PT_G && tb == PT_G) { n.kind = NK_GGG; n.ch[0] = ca[i]; n.ch[1] = cb[j]; }
                    else if (ptype == PT_G && ta == PT_B && tb == PT_Q && la == lb) { n.kind = NK_QQG_G; n.ch[0] = ca[i]; n.ch[1] = cb[j]; }
                    else if (ptype == PT_G && ta == PT_Q && tb == PT_B && la == lb) { n.kind = NK_QQG_G; n.ch[0] = cb[j]; n.ch[1] = ca[i]; }
                    else if (ptype == PT_Q && ta == PT_Q && tb == PT_G && la == line) { n.kind = NK_QG_Q; n.ch[0] = ca[i]; n.ch[1] = cb[j]; }
                    else if (ptype == PT_Q && ta == PT_G && tb == PT_Q && lb == line) { n.kind = NK_QG_Q; n.ch[0] = cb[j]; n.ch[1] = ca[i]; }
                    else if (ptype == PT_B && ta == PT_B && tb == PT_G && la == line) { n.kind = NK_BG_B; n.ch[0] = ca[i]; n.ch[1] = cb[j]; }
                    else if (ptype == PT_B && ta == PT_G && tb == PT_B && lb == line) { n.kind = NK_BG_B; n.ch[0] = cb[j]; n.ch[1] = ca[i]; }
                    else continue;
                    out.push_back(add(n));
                }
            }
            // three-way splits (gggg): A holds the lowest leg, B the lowest of the rest
            if (ptype == PT_G)
                for (unsigned A = (S - 1) & S; A; A = (A - 1) & S) {
                    if (!(A & low)) continue;
                    const unsigned R = S & ~A;
                    if ((R & (R - 1)) == 0) continue;
                    const unsigned lowR = R & (~R + 1u);
                    for (unsigned B = (R - 1) & R; B; B = (B - 1) & R) {
                        if (!(B & lowR)) continue;
                        const unsigned C = R & ~B;
                        int ta, la, tb, lb, tc, lc; classify(A, ta, la); classify(B, tb, lb); classify(C, tc, lc);
                        if (ta != PT_G || tb != PT_G || tc != PT_G) continue;
                        const std::vector<int> ca = currents(A), cb = currents(B), cc = currents(C);
                        for (size_t i = 0; i < ca.size(); ++i) for (size_t j = 0; j < cb.size(); ++j) for (size_t k = 0; k < cc.size(); ++k)
                            for (int piece = 0; piece < 3; ++piece) {
                                Node n; n.ptype = PT_G; n.line = -1; n.mask = S; n.kind = NK_GGGG; n.piece = piece; n.leg = -1; n.pairing = ip;
                                n.ch[0] = ca[i]; n.ch[1] = cb[j]; n.ch[2] = cc[k];
                                n.n_topo_weight = D.nodes[ca[i]].n_topo_weight * D.nodes[cb[j]].n_topo_weight * D.nodes[cc[k]].n_topo_weight / 3.0;
                                out.push_back(add(n));
                            }
                    }
                }
        }
        memo[S] = out;
        return memo[S];
    }
private:
    int add(const Node& n) { D.nodes.push_back(n); return (int)D.nodes.size() - 1; }
    DiagramSet& D;
    const Pairing& pr;
    int ip;
    std::map<unsigned, std::vector<int> > memo;
};

inline void enumerate_diagrams(const Process& P, DiagramSet& D) {
    D.proc = P;
    D.pairings = enumerate_pairings(P);
    D.root = P.n_ext() - 1;
    D.n_topologies = 0.0;
    const unsigned all = (1u << P.n_ext()) - 1u;
    const unsigned S = all & ~(1u << D.root);
    for (size_t ip = 0; ip < D.pairings.size(); ++ip) {
        Enumerator en(D, (int)ip);
        int ptype, line; en.classify(S, ptype, line);
        // the subtree must deliver the particle that the root leg absorbs
        const std::vector<int> c = en.currents(S);
        for (size_t i = 0; i < c.size(); ++i) {
            const Node& n = D.nodes[c[i]];
            const Leg& R = P.legs[D.root];
            bool ok = false;
            if (R.kind == LEG_G) ok = (n.ptype == PT_G);
            else if (R.kind == LEG_OUT) ok = (n.ptype == PT_Q && n.line == D.pairings[ip].line_of_leg[D.root]);
            else ok = (n.ptype == PT_B && n.line == D.pairings[ip].line_of_leg[D.root]);
            if (!ok) continue;
            D.diagrams.push_back(c[i]);
            D.diagram_sign.push_back(D.pairings[ip].sign);
            D.n_topologies += n.n_topo_weight;
        }
    }
}
}  // namespace orc
