// heget-b200 process generator, part 2: process description, off-shell current graph, diagram closings,
// colour basis and colour matrix.
//
// PAPER.md:77 (eq. 7): M = sum over all Feynman diagrams; PAPER.md:81 (eq. 8): M = sum_alpha T_alpha J_alpha;
// PAPER.md:87 (eq. 9): colour matrix.  MadGraph did this for the paper; here the generator does it.
//
// Method: every off-shell line of a tree diagram carries the set S of external legs behind it.  cur(S) lists every
// distinct sub-tree ("current") over S, built once from the currents of the 2- and 3-way splits of S (qqg, ggg, gggg
// vertices; a gggg vertex yields three currents, one per colour structure of eq. 40, PAPER.md:388 -- the counting
// convention of Table 1).  A diagram is an AMPLITUDE call (iovxx0 / vvvxxx / ggggxx) on three or four
// currents whose leg sets partition all legs.  The part that holds the root leg r (the last gluon) is either r alone or,
// when the other side of a cubic root vertex would be a single leg i, the two-leg current over {i, r}: this re-rooting
// means no current over more than n-3 legs is ever needed.
#pragma once
#include <string>
#include <sstream>
#include <set>
#include "colour.hpp"

namespace heget {

enum LegType { LEG_G = 0, LEG_QIN = 1, LEG_QOUT = 2 };   // QIN: the fermion arrow enters the diagram (initial q, final q~)
struct Leg { int type; int flavour; bool initial; bool anti; };

struct Process {
    std::string name;
    std::vector<Leg> legs;
    int n;
    double sym_factor, avg_color, avg_spin;      // 1/prod k!, 1/(n_a n_b), 1/4
};

static inline Process parse_process(const std::string& text) {
    Process P; P.name = text;
    std::istringstream in(text);
    std::string tok; bool fin = false;
    std::map<std::string, int> mult;
    while (in >> tok) {
        if (tok == ">" || tok == "->") { if (fin) throw std::runtime_error("two arrows in process"); fin = true; continue; }
        Leg L; L.initial = !fin; L.anti = false; L.flavour = -1;
        if (tok == "g") L.type = LEG_G;
        else {
            std::string f = tok;
            if (f.size() > 1 && f[f.size() - 1] == '~') { L.anti = true; f.erase(f.size() - 1); }
            const std::string names = "udscb";
            if (f.size() != 1 || names.find(f) == std::string::npos) throw std::invalid_argument("unsupported particle '" + tok + "'");
            L.flavour = (int)names.find(f);
            L.type = (L.initial != L.anti) ? LEG_QIN : LEG_QOUT;
        }
        if (fin) mult[tok] += 1;
        P.legs.push_back(L);
    }
    P.n = (int)P.legs.size();
    int ninit = 0; for (int i = 0; i < P.n; ++i) ninit += P.legs[i].initial;
    if (!fin || ninit != 2) throw std::runtime_error("process must read 'a b > c d ...'");
    if (P.n < 4) throw std::runtime_error("need at least a 2 -> 2 process");
    P.sym_factor = 1.0;
    for (std::map<std::string, int>::iterator it = mult.begin(); it != mult.end(); ++it) for (int k = 2; k <= it->second; ++k) P.sym_factor /= k;
    P.avg_color = 1.0 / ((P.legs[0].type == LEG_G ? 8.0 : 3.0) * (P.legs[1].type == LEG_G ? 8.0 : 3.0));
    P.avg_spin = 0.25;
    return P;
}

enum PType { PT_G = 0, PT_F = 1, PT_B = 2 };                      // gluon, psi (holds an in-end), psibar (holds an out-end)
enum CKind { CK_LEAF = 0, CK_GGG, CK_GGGG, CK_FUSE, CK_FG, CK_BG, CK_OPEN3, CK_OPEN4, CK_SUM };   // OPEN*: vertex with one leg left open, no propagator // jvvxx0, jgggx0, jioxx0, fvixx0, fvoxx0

// one vertex evaluation inside a merged current (CK_SUM): coef * vertex_kind(ch...) ; the propagator is applied to the sum
struct Term { int kind, ch[3], piece; Frac coef; };

struct Cur {
    int id; unsigned mask; int size;
    int ptype, end_leg;               // F: in-end leg, B: out-end leg, G: -1
    int kind, ch[3], piece, leg;
    std::vector<std::pair<int, int> > pairs;   // completed quark lines (in-end, out-end) inside
    unsigned varmask;                 // legs whose helicity/chirality bit selects the variant
    CExpr colour;
    std::vector<Term> terms;          // CK_SUM only
    double n_diag, n_topo;            // Feynman sub-diagrams summed in this current (Table 1 convention / plain topologies)
};

enum AKind { AK_VVV = 0, AK_GGGG, AK_IOV, AK_DOT };   // DOT: (open vertex, wavefunction) Minkowski product
struct Closing {
    int kind, piece;
    int c[4];                         // current ids; AK_IOV: (psibar, psi, gluon)
    std::vector<std::pair<int, int> > pairs;
    int fermi_sign;
    std::vector<std::pair<int, Frac> > coef;   // (basis index alpha, coefficient): eq. 8
    double topo_weight;
};

struct Graph {
    Process P;
    int root;
    bool paper_basis;
    // merge = true: currents over the same legs whose colour factors are proportional (a four-gluon piece and the pair of
    // three-gluon vertices with the same f.f structure, eq. 36/40) are summed into ONE stored current
    // (kind CK_SUM, one Term per vertex evaluation).  By linearity of every vertex in each of its legs the sum over diagrams
    // (eq. 7) is unchanged; the parents and closings are then built from the merged currents only.
    bool merge = false;
    // centroid = true: diagrams are closed at their centroid vertex, so no current over more than n/2 legs is needed
    // (default: at the vertex of the root leg, re-rooted when the other side of a cubic root vertex is a single leg: <= n-3 legs)
    bool centroid = false;
    double n_diagrams_paper = 0;
    ColourAlgebra ca;
    std::vector<Cur> cur;
    std::map<unsigned, std::vector<int> > by_mask;
    std::vector<Closing> closings;
    std::vector<CTerm> basis;
    std::vector<Frac> C;              // m x m exact colour matrix, WITHOUT 1/(n_a n_b)  (eq. 9)
    int n_lines;
    double n_topologies;

    int popcount(unsigned m) const { int c = 0; while (m) { c += m & 1u; m >>= 1; } return c; }

    int add(const Cur& c) { cur.push_back(c); cur.back().id = (int)cur.size() - 1; by_mask[c.mask].push_back(cur.back().id); return cur.back().id; }

    // combine the children at one vertex; returns false if no vertex exists
    bool combine(const std::vector<int>& ch, Cur& out, int piece) {
        out.kind = -1; out.piece = piece; out.leg = -1; out.ch[0] = out.ch[1] = out.ch[2] = -1;
        out.mask = 0; out.pairs.clear(); out.varmask = 0;
        for (size_t i = 0; i < ch.size(); ++i) {
            const Cur& c = cur[ch[i]];
            out.mask |= c.mask; out.varmask |= c.varmask;
            out.pairs.insert(out.pairs.end(), c.pairs.begin(), c.pairs.end());
        }
        out.size = popcount(out.mask);
        if (ch.size() == 3) {
            for (int i = 0; i < 3; ++i) if (cur[ch[i]].ptype != PT_G) return false;
            out.kind = CK_GGGG; out.ptype = PT_G; out.end_leg = -1;
            for (int i = 0; i < 3; ++i) out.ch[i] = ch[i];
            return true;
        }
        const Cur& a = cur[ch[0]]; const Cur& b = cur[ch[1]];
        if (a.ptype == PT_G && b.ptype == PT_G) { out.kind = CK_GGG; out.ptype = PT_G; out.end_leg = -1; out.ch[0] = ch[0]; out.ch[1] = ch[1]; return true; }
        if ((a.ptype == PT_B && b.ptype == PT_F) || (a.ptype == PT_F && b.ptype == PT_B)) {
            const Cur& B = a.ptype == PT_B ? a : b; const Cur& F = a.ptype == PT_B ? b : a;
            if (P.legs[B.end_leg].flavour != P.legs[F.end_leg].flavour) return false;
            out.kind = CK_FUSE; out.ptype = PT_G; out.end_leg = -1; out.ch[0] = B.id; out.ch[1] = F.id;
            out.pairs.push_back(std::make_pair(F.end_leg, B.end_leg));
            // the line's chirality is read from its in-end bit; the out-end bit must agree (checked per thread)
            out.varmask &= ~(1u << B.end_leg);
            return true;
        }
        if ((a.ptype == PT_F && b.ptype == PT_G) || (a.ptype == PT_G && b.ptype == PT_F)) {
            const Cur& F = a.ptype == PT_F ? a : b; const Cur& G = a.ptype == PT_F ? b : a;
            out.kind = CK_FG; out.ptype = PT_F; out.end_leg = F.end_leg; out.ch[0] = F.id; out.ch[1] = G.id; return true;
        }
        if ((a.ptype == PT_B && b.ptype == PT_G) || (a.ptype == PT_G && b.ptype == PT_B)) {
            const Cur& B = a.ptype == PT_B ? a : b; const Cur& G = a.ptype == PT_B ? b : a;
            out.kind = CK_BG; out.ptype = PT_B; out.end_leg = B.end_leg; out.ch[0] = B.id; out.ch[1] = G.id; return true;
        }
        return false;
    }

    void colour_of(Cur& c) {
        switch (c.kind) {
        case CK_GGG:  c.colour = ca.join3(cur[c.ch[0]].colour, cur[c.ch[1]].colour); break;
        case CK_GGGG: c.colour = ca.join4(cur[c.ch[0]].colour, cur[c.ch[1]].colour, cur[c.ch[2]].colour, c.piece); break;
        case CK_FUSE: c.colour = ca.fuse_gluon(cur[c.ch[0]].colour, cur[c.ch[1]].colour); break;
        case CK_FG:   c.colour = ca.attach(cur[c.ch[0]].colour, cur[c.ch[1]].colour, true); break;
        case CK_BG:   c.colour = ca.attach(cur[c.ch[0]].colour, cur[c.ch[1]].colour, false); break;
        default: break;
        }
    }

    // all ways to split S into k unordered non-empty parts (part holding the lowest leg first, then recursively)
    static void splits(unsigned S, int k, std::vector<std::vector<unsigned> >& out) {
        if (k == 1) { out.push_back(std::vector<unsigned>(1, S)); return; }
        const unsigned low = S & (~S + 1u);
        for (unsigned A = (S - 1) & S; A; A = (A - 1) & S) {
            if (!(A & low)) continue;
            std::vector<std::vector<unsigned> > rest;
            splits(S & ~A, k - 1, rest);
            for (size_t i = 0; i < rest.size(); ++i) { std::vector<unsigned> v(1, A); v.insert(v.end(), rest[i].begin(), rest[i].end()); out.push_back(v); }
        }
    }

    const std::vector<int>& currents(unsigned S) {
        std::map<unsigned, std::vector<int> >::iterator it = by_mask.find(S);
        if (it != by_mask.end()) return it->second;
        by_mask[S] = std::vector<int>();
        if (popcount(S) == 1) {
            int leg = 0; while (!((S >> leg) & 1u)) ++leg;
            Cur c; c.mask = S; c.size = 1; c.kind = CK_LEAF; c.leg = leg; c.piece = 0; c.ch[0] = c.ch[1] = c.ch[2] = -1; c.varmask = S;
            const Leg& L = P.legs[leg];
            if (L.type == LEG_G) { c.ptype = PT_G; c.end_leg = -1; c.colour = ca.leaf_gluon(leg); }
            else if (L.type == LEG_QIN) { c.ptype = PT_F; c.end_leg = leg; c.colour = ca.leaf_psi(leg); }
            else { c.ptype = PT_B; c.end_leg = leg; c.colour = ca.leaf_psibar(leg); }
            c.n_diag = 1.0; c.n_topo = 1.0;
            add(c);
            return by_mask[S];
        }
        std::vector<Cur> raws;
        for (int k = 2; k <= 3; ++k) {
            std::vector<std::vector<unsigned> > sp; splits(S, k, sp);
            for (size_t s = 0; s < sp.size(); ++s) {
                std::vector<std::vector<int> > lists;
                bool empty = false;
                for (int j = 0; j < k; ++j) { lists.push_back(currents(sp[s][j])); if (lists.back().empty()) empty = true; }
                if (empty) continue;
                std::vector<size_t> idx(k, 0);
                for (;;) {
                    std::vector<int> ch(k); for (int j = 0; j < k; ++j) ch[j] = lists[j][idx[j]];
                    for (int piece = 0; piece < (k == 3 ? 3 : 1); ++piece) {
                        Cur c;
                        if (combine(ch, c, piece)) {
                            colour_of(c);
                            c.n_diag = 1.0; c.n_topo = (c.kind == CK_GGGG) ? 1.0 / 3.0 : 1.0;
                            for (int q = 0; q < 3; ++q) if (c.ch[q] >= 0) { c.n_diag *= cur[c.ch[q]].n_diag; c.n_topo *= cur[c.ch[q]].n_topo; }
                            if (merge) raws.push_back(c); else add(c);
                        }
                    }
                    int j = k - 1; while (j >= 0 && ++idx[j] == lists[j].size()) { idx[j] = 0; --j; }
                    if (j < 0) break;
                }
            }
        }
        if (merge) merge_raws(raws);
        return by_mask[S];
    }

    // group the raw currents over one leg set by (type, open end, completed quark lines, normalised colour) and store one
    // CK_SUM current per group; raw currents whose colour vanishes identically are dropped
    void merge_raws(std::vector<Cur>& raws) {
        typedef std::pair<std::pair<std::pair<int, int>, std::vector<std::pair<int, int> > >, CExpr> Key;
        std::map<Key, int> index;
        std::vector<int> order;
        for (size_t r = 0; r < raws.size(); ++r) {
            Cur& c = raws[r];
            if (c.colour.empty()) continue;
            std::sort(c.pairs.begin(), c.pairs.end());
            const Frac lead = c.colour.begin()->second, inv(lead.d, lead.n);
            Key key; key.first.first = std::make_pair(c.ptype, c.end_leg); key.first.second = c.pairs; key.second = scaled(c.colour, inv);
            Term t; t.kind = c.kind; t.piece = c.piece; for (int q = 0; q < 3; ++q) t.ch[q] = c.ch[q];
            std::map<Key, int>::iterator it = index.find(key);
            if (it == index.end()) {
                Cur m = c; m.kind = CK_SUM; m.ch[0] = m.ch[1] = m.ch[2] = -1; m.piece = 0; m.terms.clear();
                t.coef = Frac(1); m.terms.push_back(t);
                const int id = add(m);
                index[key] = id; order.push_back(id);
                lead_of[id] = lead;
            } else {
                Cur& m = cur[it->second];
                const Frac l0 = lead_of[it->second];
                t.coef = lead * Frac(l0.d, l0.n);
                m.terms.push_back(t); m.n_diag += c.n_diag; m.n_topo += c.n_topo;
            }
        }
    }
    std::map<int, Frac> lead_of;

    static int perm_sign(std::vector<std::pair<int, int> > pairs) {
        std::sort(pairs.begin(), pairs.end());
        int inv = 0;
        for (size_t i = 0; i < pairs.size(); ++i) for (size_t j = i + 1; j < pairs.size(); ++j) inv += pairs[i].second > pairs[j].second;
        return (inv & 1) ? -1 : +1;
    }

    void try_closing(const std::vector<int>& ch, std::map<CTerm, int>& basis_index, std::vector<CExpr>& colours) {
        const int k = (int)ch.size();
        int ng = 0, nf = 0, nb = 0;
        for (int j = 0; j < k; ++j) { const int t = cur[ch[j]].ptype; ng += t == PT_G; nf += t == PT_F; nb += t == PT_B; }
        for (int piece = 0; piece < (k == 4 ? 3 : 1); ++piece) {
            Closing cl; cl.piece = piece; cl.c[0] = cl.c[1] = cl.c[2] = cl.c[3] = -1; cl.topo_weight = (k == 4) ? 1.0 / 3.0 : 1.0;
            CExpr col;
            for (int j = 0; j < k; ++j) cl.pairs.insert(cl.pairs.end(), cur[ch[j]].pairs.begin(), cur[ch[j]].pairs.end());
            if (k == 3 && ng == 3) {
                cl.kind = AK_VVV; for (int j = 0; j < 3; ++j) cl.c[j] = ch[j];
                col = ca.amp_vvv(cur[ch[0]].colour, cur[ch[1]].colour, cur[ch[2]].colour);
            } else if (k == 4 && ng == 4) {
                cl.kind = AK_GGGG; for (int j = 0; j < 4; ++j) cl.c[j] = ch[j];
                col = ca.amp_gggg(cur[ch[0]].colour, cur[ch[1]].colour, cur[ch[2]].colour, cur[ch[3]].colour, piece);
            } else if (k == 3 && ng == 1 && nf == 1 && nb == 1) {
                int B = -1, F = -1, G = -1;
                for (int j = 0; j < 3; ++j) { const int t = cur[ch[j]].ptype; if (t == PT_B) B = ch[j]; else if (t == PT_F) F = ch[j]; else G = ch[j]; }
                if (P.legs[cur[B].end_leg].flavour != P.legs[cur[F].end_leg].flavour) return;
                cl.kind = AK_IOV; cl.c[0] = B; cl.c[1] = F; cl.c[2] = G;
                cl.pairs.push_back(std::make_pair(cur[F].end_leg, cur[B].end_leg));
                col = ca.amp_iov(cur[B].colour, cur[F].colour, cur[G].colour);
            } else return;
            for (int j = 0; j < k; ++j) for (int m2 = 0; m2 < 3; ++m2) if (cur[ch[j]].kind == CK_GGGG && false) (void)m2;
            cl.fermi_sign = perm_sign(cl.pairs);
            for (CExpr::const_iterator it = col.begin(); it != col.end(); ++it) if (!basis_index.count(it->first)) basis_index[it->first] = 0;
            colours.push_back(col);
            closings.push_back(cl);
        }
    }

    double topo_weight_of(int id) const {
        const Cur& c = cur[id];
        if (c.kind == CK_LEAF) return 1.0;
        if (c.kind == CK_SUM) return c.n_topo;
        double w = (c.kind == CK_GGGG) ? 1.0 / 3.0 : 1.0;
        for (int j = 0; j < 3; ++j) if (c.ch[j] >= 0) w *= topo_weight_of(c.ch[j]);
        return w;
    }

    void build(const Process& proc, bool paper_colour_basis) {
        P = proc; paper_basis = paper_colour_basis;
        const int n = P.n;
        if (n > 8) throw std::invalid_argument("at most 2 -> 6");
        int nin = 0, nout = 0, ngl = 0;
        for (int i = 0; i < n; ++i) { nin += P.legs[i].type == LEG_QIN; nout += P.legs[i].type == LEG_QOUT; ngl += P.legs[i].type == LEG_G; }
        if (nin != nout) throw std::invalid_argument("quark number is not conserved");
        n_lines = nin;
        if (n_lines > 2) throw std::invalid_argument("at most two quark lines");
        ca.keep_bridge = paper_basis && n_lines == 2;
        root = n - 1;
        for (int i = n - 1; i >= 0; --i) if (P.legs[i].type == LEG_G) { root = i; break; }
        const unsigned all = (1u << n) - 1u, rbit = 1u << root, rest = all & ~rbit;
        std::map<CTerm, int> basis_index;
        std::vector<CExpr> colours;
        const int max_part = std::max(1, n - 3);
        if (centroid) {
            // every tree has a vertex all of whose branches hold at most n/2 legs; when a branch holds exactly n/2 the vertex
            // at its other end qualifies too, and the one on the root's side is taken: each diagram is closed exactly once
            for (int k = 3; k <= 4; ++k) {
                std::vector<std::vector<unsigned> > sp; splits(all, k, sp);
                for (size_t s = 0; s < sp.size(); ++s) {
                    bool ok = true;
                    for (int j = 0; j < k; ++j) { const int sz = popcount(sp[s][j]); if (2 * sz > n || (2 * sz == n && (sp[s][j] & rbit))) ok = false; }
                    if (!ok) continue;
                    std::vector<unsigned> parts(sp[s].begin(), sp[s].end() - 1);
                    close_parts(parts, sp[s].back(), basis_index, colours);
                }
            }
        } else {
        // (i) the root alone + a 2- or 3-way split of the other legs, every part <= n-3 legs
        for (int k = 2; k <= 3; ++k) {
            std::vector<std::vector<unsigned> > sp; splits(rest, k, sp);
            for (size_t s = 0; s < sp.size(); ++s) {
                bool ok = true; for (int j = 0; j < k; ++j) if (popcount(sp[s][j]) > max_part) ok = false;
                if (!ok) continue;
                close_parts(sp[s], rbit, basis_index, colours);
            }
        }
        // (ii) re-rooted: the two-leg current over {i, root} + a split of the remaining n-2 legs
        if (n >= 4) for (int i = 0; i < n; ++i) if (i != root) {
            const unsigned pair = rbit | (1u << i), others = all & ~pair;
            if (n - 2 == 1) continue;
            for (int k = 2; k <= 3; ++k) {
                if (popcount(others) < k) continue;
                std::vector<std::vector<unsigned> > sp; splits(others, k, sp);
                for (size_t s = 0; s < sp.size(); ++s) close_parts(sp[s], pair, basis_index, colours);
            }
        }
        }
        if (closings.empty()) throw std::invalid_argument("no tree-level QCD diagram for this process");
        // basis = every distinct colour structure that occurs (single traces / quark strings), in canonical order
        int m = 0;
        for (std::map<CTerm, int>::iterator it = basis_index.begin(); it != basis_index.end(); ++it) { it->second = m++; basis.push_back(it->first); }
        n_topologies = 0.0;
        for (size_t l = 0; l < closings.size(); ++l) {
            Closing& cl = closings[l];
            for (CExpr::const_iterator it = colours[l].begin(); it != colours[l].end(); ++it)
                cl.coef.push_back(std::make_pair(basis_index[it->first], it->second * Frac(cl.fermi_sign)));
            double w = cl.topo_weight, nd = 1.0; for (int j = 0; j < 4; ++j) if (cl.c[j] >= 0) { w *= topo_weight_of(cl.c[j]); nd *= cur[cl.c[j]].n_diag; }
            n_topologies += w; n_diagrams_paper += nd;
        }
        std::vector<int> gl; for (int i = 0; i < n; ++i) if (P.legs[i].type == LEG_G) gl.push_back(i);
        C.assign((size_t)m * m, Frac(0));
        for (int a = 0; a < m; ++a) for (int b = a; b < m; ++b) { Frac v = ca.overlap(basis[a], basis[b], gl); C[(size_t)a * m + b] = v; C[(size_t)b * m + a] = v; }
    }

    void close_parts(const std::vector<unsigned>& parts, unsigned root_part, std::map<CTerm, int>& basis_index, std::vector<CExpr>& colours) {
        std::vector<unsigned> all_parts = parts; all_parts.push_back(root_part);
        std::sort(all_parts.begin(), all_parts.end(), [](unsigned a, unsigned b) { return (a & (~a + 1u)) < (b & (~b + 1u)); });
        const int k = (int)all_parts.size();
        std::vector<std::vector<int> > lists;
        for (int j = 0; j < k; ++j) { lists.push_back(currents(all_parts[j])); if (lists.back().empty()) return; }
        std::vector<size_t> idx(k, 0);
        for (;;) {
            std::vector<int> ch(k); for (int j = 0; j < k; ++j) ch[j] = lists[j][idx[j]];
            try_closing(ch, basis_index, colours);
            int j = k - 1; while (j >= 0 && ++idx[j] == lists[j].size()) { idx[j] = 0; --j; }
            if (j < 0) break;
        }
    }
};
}  // namespace heget
