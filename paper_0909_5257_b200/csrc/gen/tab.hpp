// heget-b200 process generator, part 4: the TABLE program of a process -- the data the generic kernels of
// csrc/device/heget_tab.cuh interpret (steps a3-a8 of SURVEY.md 8(a); eqs. 4, 7-12 of the paper).
//
// Why a second back end.  The straight-line kernels of emit.hpp put one helicity configuration of gg -> 4g / u u~ -> 5g into
// 60 k - 180 k instructions: 1-3 MB of code against a ~128 kB instruction cache, instruction-fetch bound (round-1 profiles).
// Here the diagram chain is DATA: the kernel is a few kB of loops over tables, and three reorganisations of the same sum
// over Feynman diagrams (eq. 7) cut the arithmetic itself:
//   1. merged currents (graph.hpp, Graph::merge): sub-currents over the same legs with proportional colour factors are
//      summed into one stored current (every vertex is linear in each leg);
//   2. centroid closings (Graph::centroid): each diagram is closed at its centroid vertex, so no current spans more than
//      n/2 legs (u u~ -> 5g: 133 currents and 1350 closings instead of 397 and 1890);
//   3. helicity recycling: a current over the leg set S depends only on the helicities of the legs in S, so it is computed
//      once per 2^|S| helicity assignment ("variant") per event and not once per full configuration (SURVEY.md 8(d),
//      "factorised" scheme); only the closing amplitudes, J (eq. 8) and the colour form (eq. 10) are per configuration.
// Closings whose colour coefficient vectors c_{alpha l} are proportional form a group; a group's amplitudes are summed in a
// register and J is touched once per group (eq. 8 read as J = sum_g k_g S_g).  When the group vectors span fewer dimensions
// than the merged colour basis (pure-gluon processes: the f-basis identities), J is accumulated on a basis of that span and
// the colour matrix is the exact congruence B^T C B.
#pragma once
#include <cstdint>
#include <cstring>
#include "emit.hpp"
#include "tabprog.hpp"

namespace heget {

struct TabBuilder {
    struct OpT { int kind, ch[3]; Frac coef; };
    const Graph& G;            // built with merge (and usually centroid)
    Emitter E;
    TabProgram P;
    std::vector<int> base32, lognv;      // per current
    std::map<unsigned, int> kslot;
    std::vector<int> chisign;            // per leg: chirality = chisign * helicity for quark legs

    TabBuilder(const Graph& g, const std::string& tag) : G(g), E(g, tag, EmitOptions()) {}

    static int popc(unsigned m) { int c = 0; while (m) { c += m & 1u; m >>= 1; } return c; }
    static unsigned deposit(unsigned v, unsigned mask) { unsigned r = 0; int k = 0; for (int i = 0; i < 32; ++i) if ((mask >> i) & 1u) { if ((v >> k) & 1u) r |= 1u << i; ++k; } return r; }
    static unsigned extract(unsigned bits, unsigned mask) { unsigned r = 0; int k = 0; for (int i = 0; i < 32; ++i) if ((mask >> i) & 1u) { if ((bits >> i) & 1u) r |= 1u << k; ++k; } return r; }
    int hel_of_bit(unsigned bits, int leg) const { return ((bits >> leg) & 1u) ? +1 : -1; }
    int chi_of_leg(unsigned bits, int leg) const { return chisign[leg] * hel_of_bit(bits, leg); }
    // helicity bits of every leg behind current c for its variant v (out-ends of completed quark lines follow their in-ends)
    // Legs whose helicity is the same in every evaluated configuration (leg 0 after parity folding; both ends of the quark line of
    // u u~ -> n g) select nothing: they are left out of the variant index, which halves the variants of every current that holds them.
    unsigned constmask = 0, constbits = 0;
    unsigned vm(const Cur& c) const { return c.varmask & ~constmask; }
    unsigned pattern(const Cur& c, unsigned v) const {
        unsigned p = deposit(v, vm(c)) | constbits;
        for (size_t q = 0; q < c.pairs.size(); ++q) {
            const int in = c.pairs[q].first, oe = c.pairs[q].second;
            if (((c.varmask | constmask) >> oe) & 1u) continue;
            const int h = chi_of_leg(p, in) * chisign[oe];
            if (h > 0) p |= 1u << oe; else p &= ~(1u << oe);
        }
        return p;
    }
    int slot_of(unsigned mask) { std::map<unsigned, int>::iterator it = kslot.find(mask); if (it != kslot.end()) return it->second; const int s = (int)kslot.size(); kslot[mask] = s; return s; }

    // ---- rank reduction of the group vectors (exact) -----------------------------------------------------------------
    // groups g have vectors v_g in Q^NJ (E.group_key).  Returns basis group ids and X[g] = sparse coefficients on that basis.
    bool reduce_rank(const std::vector<int>& order, std::vector<int>& basis, std::vector<std::vector<std::pair<int, Frac> > >& X) const {
        const int ng = (int)E.group_key.size(), NJ = E.NJ;
        struct Row { std::vector<Frac> v; std::vector<Frac> comb; int pivot; };
        std::vector<Row> rows;
        basis.clear(); X.assign(ng, std::vector<std::pair<int, Frac> >());
        for (int oi = 0; oi < ng; ++oi) {
            const int g = order[oi];
            std::vector<Frac> v(NJ, Frac(0)), comb;      // v_g - sum t_k row_k ; comb = coefficients on the basis vectors b_j
            for (size_t t = 0; t < E.group_key[g].size(); ++t) v[E.group_key[g][t].first] = E.group_key[g][t].second;
            comb.assign(basis.size(), Frac(0));
            for (size_t k = 0; k < rows.size(); ++k) {
                const Frac t = v[rows[k].pivot];
                if (t.zero()) continue;
                for (int a = 0; a < NJ; ++a) if (!rows[k].v[a].zero()) v[a] = v[a] - t * rows[k].v[a];
                for (size_t j = 0; j < rows[k].comb.size(); ++j) if (!rows[k].comb[j].zero()) comb[j] = comb[j] + t * rows[k].comb[j];
            }
            int piv = -1; for (int a = 0; a < NJ; ++a) if (!v[a].zero()) { piv = a; break; }
            if (piv < 0) {
                for (size_t j = 0; j < comb.size(); ++j) if (!comb[j].zero()) X[g].push_back(std::make_pair((int)j, comb[j]));
            } else {
                // new basis vector b_new = v_g; echelon row = (v_g - sum t_k row_k) / pivot value, fully reduced rows
                const int id = (int)basis.size(); basis.push_back(g);
                Row r; r.pivot = piv; r.v = v; r.comb.assign(id + 1, Frac(0));
                for (size_t j = 0; j < comb.size(); ++j) r.comb[j] = -comb[j];
                r.comb[id] = Frac(1);
                const Frac inv(v[piv].d, v[piv].n);
                for (int a = 0; a < NJ; ++a) r.v[a] = r.v[a] * inv;
                for (size_t j = 0; j < r.comb.size(); ++j) r.comb[j] = r.comb[j] * inv;
                // eliminate the new pivot from the older rows (keeps every row reduced, so one pass suffices above)
                for (size_t k = 0; k < rows.size(); ++k) {
                    const Frac t = rows[k].v[piv];
                    if (t.zero()) continue;
                    for (int a = 0; a < NJ; ++a) if (!r.v[a].zero()) rows[k].v[a] = rows[k].v[a] - t * r.v[a];
                    rows[k].comb.resize(id + 1, Frac(0));
                    for (size_t j = 0; j < r.comb.size(); ++j) if (!r.comb[j].zero()) rows[k].comb[j] = rows[k].comb[j] - t * r.comb[j];
                }
                rows.push_back(r);
                X[g].push_back(std::make_pair(id, Frac(1)));
            }
        }
        // exact check: v_g == sum_k X[g][k] v_{basis[k]}
        for (int g = 0; g < ng; ++g) {
            std::vector<Frac> v(NJ, Frac(0));
            for (size_t t = 0; t < X[g].size(); ++t) { const int b = basis[X[g][t].first]; for (size_t q = 0; q < E.group_key[b].size(); ++q) v[E.group_key[b][q].first] = v[E.group_key[b][q].first] + X[g][t].second * E.group_key[b][q].second; }
            for (size_t q = 0; q < E.group_key[g].size(); ++q) v[E.group_key[g][q].first] = v[E.group_key[g][q].first] - E.group_key[g][q].second;
            for (int a = 0; a < NJ; ++a) if (!v[a].zero()) return false;
        }
        return true;
    }

    static void put4(std::vector<uint32_t>& v, uint32_t a, uint32_t b, uint32_t c, uint32_t d) { v.push_back(a); v.push_back(b); v.push_back(c); v.push_back(d); }
    // rational coefficients live once, as doubles, in a pool; the tables hold indices (a float would round 1/3)
    std::map<std::pair<long long, long long>, uint32_t> coef_index;
    uint32_t coef_of(const Frac& f) {
        const std::pair<long long, long long> key(f.n, f.d);
        std::map<std::pair<long long, long long>, uint32_t>::iterator it = coef_index.find(key);
        if (it != coef_index.end()) return it->second;
        const uint32_t id = (uint32_t)P.coef.size(); P.coef.push_back(f.value()); coef_index[key] = id; return id;
    }

    bool fold_parity = true, const_legs = true;
    void build(const Graph* paper, bool allow_rank_reduction = true) {
        const int n = G.P.n;
        P.name = G.P.name; P.tag = E.tag; P.n_ext = n; P.n_hel = 1 << n;
        P.sym_factor = G.P.sym_factor; P.avg_color = G.P.avg_color; P.avg_spin = G.P.avg_spin;
        chisign.assign(n, 0);
        for (int i = 0; i < n; ++i) if (G.P.legs[i].type != LEG_G) chisign[i] = G.P.legs[i].anti ? +1 : -1;      // Emitter::chi_of: chi = -h (anti: +h)
        E.analyse_helicities(); E.reduce_colour(); E.build_groups();
        P.n_gluons = E.ng; P.n_quark_legs = E.nq; P.NJ = E.NJ;
        // Parity folding of the helicity sum (eq. 12): QCD conserves parity, so |M|^2 of a configuration equals that of the
        // configuration with every helicity flipped (the oracle pins this per configuration, tests/test_oracle_amplitudes.py).
        // The non-vanishing configurations come in such pairs; one of each pair (leg 0 at helicity -1) is evaluated and counted
        // twice.  HEL_FIXED / HEL_SAMPLE map a requested configuration onto its evaluated partner.
        std::vector<int> kept;
        for (int h = 0; h < E.NH; ++h) if (!fold_parity || E.hel_of(h)[0] < 0) kept.push_back(h);
        if (fold_parity && 2 * (int)kept.size() != E.NH) throw std::runtime_error("helicity configurations are not closed under parity");
        P.NH = (int)kept.size(); P.n_hel_nonzero = E.NH; P.hel_weight = fold_parity ? 2 : 1;
        {
            unsigned all1 = (1u << n) - 1u, all0 = (1u << n) - 1u;      // legs at +1 (at -1) in every evaluated configuration
            for (size_t q = 0; q < kept.size(); ++q) { const std::vector<int> hv = E.hel_of(kept[q]); unsigned b = 0; for (int i = 0; i < n; ++i) if (hv[i] > 0) b |= 1u << i; all1 &= b; all0 &= ~b; }
            constmask = const_legs ? (all1 | all0) : 0u; constbits = const_legs ? all1 : 0u;
        }
        P.nchunks = (P.NH + 31) / 32; P.cpc = (P.NH + P.nchunks - 1) / P.nchunks;
        P.n_diagrams = (int)std::lround(G.n_diagrams_paper); P.n_topologies = (int)std::lround(G.n_topologies);
        const Graph& GP = paper ? *paper : G;
        P.n_color = (int)GP.basis.size(); P.n_color_eval = (int)G.basis.size();
        for (size_t a = 0; a < GP.C.size(); ++a) P.colour_paper.push_back(GP.C[a].value());
        for (size_t a = 0; a < E.Cred.size(); ++a) P.colour_red.push_back(E.Cred[a].value());

        // ---- J basis: the span of the group vectors ------------------------------------------------------------------
        const int ng = (int)E.group_key.size();
        P.n_groups = ng;
        std::vector<int> basis; std::vector<std::vector<std::pair<int, Frac> > > X;
        bool reduced = false;
        if (allow_rank_reduction) {
            // sparse vectors first: they make the sparsest basis; a few deterministic re-orderings are tried and the one with
            // the fewest update coefficients is kept
            std::vector<int> best_basis; std::vector<std::vector<std::pair<int, Frac> > > bestX; long best_nnz = -1;
            for (int trial = 0; trial < 8; ++trial) {
                std::vector<int> order(ng); for (int g = 0; g < ng; ++g) order[g] = g;
                unsigned long long rng = 0x9E3779B97F4A7C15ull * (trial + 1);
                if (trial > 0) for (int g = ng - 1; g > 0; --g) { rng = rng * 6364136223846793005ull + 1442695040888963407ull; std::swap(order[g], order[(rng >> 33) % (g + 1)]); }
                std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return E.group_key[a].size() < E.group_key[b].size(); });
                std::vector<int> b; std::vector<std::vector<std::pair<int, Frac> > > x;
                bool ok = false;
                try { ok = reduce_rank(order, b, x); } catch (...) { ok = false; }
                if (!ok) continue;
                long nnz = 0; bool small = true;
                for (int g = 0; g < ng; ++g) { nnz += (long)x[g].size(); for (size_t t = 0; t < x[g].size(); ++t) if (std::llabs(x[g][t].second.n) > 64 || x[g][t].second.d > 64) small = false; }
                if (!small) continue;
                if (best_nnz < 0 || nnz < best_nnz) { best_nnz = nnz; best_basis = b; bestX = x; }
            }
            long nnz0 = 0; for (int g = 0; g < ng; ++g) nnz0 += (long)E.group_key[g].size();
            if (best_nnz >= 0 && ((int)best_basis.size() < E.NJ || best_nnz < nnz0)) { basis = best_basis; X = bestX; reduced = true; }
        }
        if (reduced) {
            P.R = (int)basis.size();
            // C_acc = B^T C_red B, exact
            std::vector<Frac> CB((size_t)E.NJ * P.R, Frac(0));
            for (int k = 0; k < P.R; ++k) for (size_t q = 0; q < E.group_key[basis[k]].size(); ++q) {
                const int b = E.group_key[basis[k]][q].first; const Frac w = E.group_key[basis[k]][q].second;
                for (int a = 0; a < E.NJ; ++a) if (!E.Cred[(size_t)a * E.NJ + b].zero()) CB[(size_t)a * P.R + k] = CB[(size_t)a * P.R + k] + E.Cred[(size_t)a * E.NJ + b] * w;
            }
            cacc.assign((size_t)P.R * P.R, Frac(0));
            for (int k = 0; k < P.R; ++k) for (size_t q = 0; q < E.group_key[basis[k]].size(); ++q) {
                const int a = E.group_key[basis[k]][q].first; const Frac w = E.group_key[basis[k]][q].second;
                for (int l = 0; l < P.R; ++l) if (!CB[(size_t)a * P.R + l].zero()) cacc[(size_t)k * P.R + l] = cacc[(size_t)k * P.R + l] + w * CB[(size_t)a * P.R + l];
            }
        } else {
            P.R = E.NJ; cacc = E.Cred;
            X.assign(ng, std::vector<std::pair<int, Frac> >());
            for (int g = 0; g < ng; ++g) X[g] = E.group_key[g];
        }
        P.Rpad = (P.R + 7) / 8 * 8;
        for (size_t a = 0; a < cacc.size(); ++a) P.colour_acc.push_back(cacc[a].value());
        // tiles of 8 rows, Rpad columns each (columns beyond R are zero), one more tile of zeros at the end (the kernel prefetches one block ahead)
        P.cmat.assign((size_t)(P.Rpad / 8 + 1) * P.Rpad * 8, 0.0);
        for (int t = 0; t < P.Rpad / 8; ++t) for (int b = 0; b < P.R; ++b) for (int i = 0; i < 8; ++i) {
            const int a = t * 8 + i; if (a >= P.R || b < a) continue;
            P.cmat[((size_t)t * P.Rpad + b) * 8 + i] = cacc[(size_t)a * P.R + b].value() * (b > a ? 2.0 : 1.0);
        }

        // ---- store layout: every current holds 2^|varmask| variants of 4 (gluon) or 2 (Weyl spinor) complex components ----
        const int nc = (int)G.cur.size();
        base32.assign(nc, -1); lognv.assign(nc, 0);
        std::vector<char> needed(nc, 0);
        { std::vector<int> st; for (size_t l = 0; l < G.closings.size(); ++l) for (int j = 0; j < 4; ++j) if (G.closings[l].c[j] >= 0) st.push_back(G.closings[l].c[j]);
          while (!st.empty()) { const int c = st.back(); st.pop_back(); if (needed[c]) continue; needed[c] = 1;
              const Cur& C = G.cur[c];
              if (C.kind == CK_SUM) { for (size_t t = 0; t < C.terms.size(); ++t) for (int j = 0; j < 3; ++j) if (C.terms[t].ch[j] >= 0) st.push_back(C.terms[t].ch[j]); }
              else for (int j = 0; j < 3; ++j) if (C.ch[j] >= 0) st.push_back(C.ch[j]); } }
        int top = 0, maxsize = 1;
        P.leginfo.assign(n, 0);
        for (int pass = 0; pass < 2; ++pass) for (int c = 0; c < nc; ++c) {
            const Cur& C = G.cur[c];
            if ((C.kind == CK_LEAF) != (pass == 0)) continue;
            if (!needed[c] && C.kind != CK_LEAF) continue;
            lognv[c] = popc(vm(C));
            if (lognv[c] > 5) throw std::runtime_error("a current with more than 32 helicity variants");
            top = (top + (1 << lognv[c]) - 1) & ~((1 << lognv[c]) - 1);      // base aligned to the variant count: the FP64 layout recovers the variant from the low bits
            base32[c] = top; top += (C.ptype == PT_G ? 2 : 1) << lognv[c];
            maxsize = std::max(maxsize, C.size);
            if (C.kind == CK_LEAF) {
                const Leg& L = G.P.legs[C.leg];
                const unsigned ty = L.type == LEG_G ? (L.initial ? 1u : 0u) : (C.ptype == PT_F ? 2u : 3u);
                const unsigned single = ((constmask >> C.leg) & 1u) ? (((constbits >> C.leg) & 1u) ? 2u : 1u) : 0u;      // 0: both helicities stored, 1: only -1, 2: only +1
                P.leginfo[C.leg] = ty | ((chisign[C.leg] > 0 ? 1u : 0u) << 8) | (single << 9) | ((unsigned)base32[c] << 16);
            } else { P.n_currents++; }
        }
        if (top > 65535) throw std::runtime_error("current store exceeds the 16-bit address space of the tables");
        P.store32 = top;
        for (int i = 0; i < n; ++i) slot_of(1u << i);

        // ---- phase A: bundles of (current, variant) lanes with one sequence of vertex kinds ------------------------------
        P.n_levels = 0; P.a_level.push_back(0);
        for (int size = 2; size <= maxsize; ++size) {
            std::map<std::vector<int>, std::vector<int> > by_sig;     // signature -> currents
            std::map<int, std::vector<OpT> > terms_of;
            for (int c = 0; c < nc; ++c) {
                const Cur& C = G.cur[c];
                if (C.kind == CK_LEAF || !needed[c] || C.size != size) continue;
                std::vector<OpT> ts;
                if (C.kind == CK_SUM) { for (size_t t = 0; t < C.terms.size(); ++t) ts.push_back(make_term(C.terms[t].kind, C.terms[t].ch, C.terms[t].piece, C.terms[t].coef)); }
                else ts.push_back(make_term(C.kind, C.ch, C.piece, Frac(1)));
                std::stable_sort(ts.begin(), ts.end(), [](const OpT& a, const OpT& b) { return a.kind < b.kind; });
                std::vector<int> sig; sig.push_back(C.ptype); sig.push_back(lognv[c]);
                for (size_t t = 0; t < ts.size(); ++t) sig.push_back(ts[t].kind);
                by_sig[sig].push_back(c); terms_of[c] = ts;
                P.n_terms += (int)ts.size();
            }
            for (std::map<std::vector<int>, std::vector<int> >::iterator it = by_sig.begin(); it != by_sig.end(); ++it) {
                const int ptype = it->first[0], lnv = it->first[1], nv = 1 << lnv, nt = (int)it->first.size() - 2;
                if (nt > 8) throw std::runtime_error("more than 8 vertex terms in one merged current");
                const int per = 32 / nv;
                for (size_t o0 = 0; o0 < it->second.size(); o0 += per) {
                    const int nops = (int)std::min<size_t>(per, it->second.size() - o0);
                    uint32_t kinds = 0; for (int t = 0; t < nt; ++t) kinds |= (uint32_t)it->first[2 + t] << (4 * t);
                    put4(P.a_hdr, (uint32_t)nt | ((uint32_t)ptype << 8) | ((uint32_t)P.n_bterms << 16), kinds, (uint32_t)size, 0);
                    for (int lane = 0; lane < 32; ++lane) {
                        const int oi = lane / nv; const unsigned v = lane % nv;
                        if (oi >= nops) { P.a_out.push_back(0); P.a_out.push_back(0); continue; }
                        const int c = it->second[o0 + oi];
                        P.a_out.push_back((uint32_t)(base32[c] + (int)v) | ((uint32_t)lnv << 16) | (1u << 19));
                        P.a_out.push_back((uint32_t)slot_of(G.cur[c].mask));
                    }
                    for (int t = 0; t < nt; ++t) {
                        for (int lane = 0; lane < 32; ++lane) {
                            const int oi = lane / nv; const unsigned v = lane % nv;
                            if (oi >= nops) { put4(P.a_term, 0, 0, 0, 0); continue; }
                            const int c = it->second[o0 + oi]; const Cur& C = G.cur[c];
                            const OpT& T = terms_of[c][t];
                            const unsigned pat = pattern(C, v);
                            uint32_t addr[3] = {0, 0, 0}, ln[3] = {0, 0, 0}, ks[2] = {0, 0}, chi = 0;
                            for (int j = 0; j < 3; ++j) if (T.ch[j] >= 0) {
                                const Cur& A = G.cur[T.ch[j]];
                                addr[j] = (uint32_t)(base32[T.ch[j]] + (int)extract(pat, vm(A))); ln[j] = (uint32_t)lognv[T.ch[j]];
                            }
                            if (T.kind == TA_GGG) { ks[0] = (uint32_t)slot_of(G.cur[T.ch[0]].mask); ks[1] = (uint32_t)slot_of(G.cur[T.ch[1]].mask); }
                            int line_leg = -1;
                            if (T.kind == TA_FUSE || T.kind == TA_FG) line_leg = G.cur[T.ch[0]].end_leg;      // ch[0] = psi
                            if (T.kind == TA_BG) line_leg = G.cur[T.ch[0]].end_leg;                           // ch[0] = psibar
                            if (line_leg >= 0) chi = chi_of_leg(pat, line_leg) > 0 ? 1u : 0u;
                            if (ks[0] > 255 || ks[1] > 255) throw std::runtime_error("more than 256 momentum slots");
                            put4(P.a_term, addr[0] | (addr[1] << 16), addr[2] | (ln[0] << 16) | (ln[1] << 19) | (ln[2] << 22) | (chi << 25),
                                 ks[0] | (ks[1] << 8), coef_of(T.coef));
                            P.flops_phase_a += FlopTable::of_current(T.kind == TA_GGG ? CK_GGG : T.kind == TA_GGGG ? CK_GGGG : T.kind == TA_FUSE ? CK_FUSE : CK_FG) + (nt > 1 ? (ptype == PT_G ? 8 : 4) : 0);
                        }
                        P.n_bterms++;
                    }
                    P.n_bundles++;
                }
            }
            P.a_level.push_back((uint32_t)P.n_bundles); P.n_levels++;
        }

        // ---- phase B: closings in group order -----------------------------------------------------------------------------
        // Order of the closings: group by group (a group's amplitudes add up in one register pair); groups sorted by their kind
        // signature and every other group walked backwards, so closings of one vertex kind come in runs (the kernel's uniform
        // branch on the kind then changes direction rarely).
        std::vector<int> order;
        { std::vector<std::vector<int> > of_group(ng);
          auto kind_of = [&](int l) { return G.closings[l].kind == AK_VVV ? 0 : G.closings[l].kind == AK_GGGG ? 1 : 2; };
          for (size_t l = 0; l < G.closings.size(); ++l) if (E.group_of[l] >= 0) of_group[E.group_of[l]].push_back((int)l);
          std::vector<std::pair<std::vector<int>, int> > sig(ng);
          for (int g = 0; g < ng; ++g) {
              std::stable_sort(of_group[g].begin(), of_group[g].end(), [&](int a, int b) { return kind_of(a) < kind_of(b); });
              for (size_t k = 0; k < of_group[g].size(); ++k) sig[g].first.push_back(kind_of(of_group[g][k]));
              sig[g].second = g;
          }
          std::stable_sort(sig.begin(), sig.end(), [](const std::pair<std::vector<int>, int>& a, const std::pair<std::vector<int>, int>& b) { return a.first < b.first; });
          // ... and the sorted sequence is walked from both ends in turn (first, last, second, ...): the groups with many closings and
          // few colour updates sit at one end and the single-closing groups with up to eight updates at the other, and a
          // warp-specialised launch (heget_tab.cuh) wants the work of its producer warps and of its updater warp mixed evenly in time
          { std::vector<std::pair<std::vector<int>, int> > mixed; mixed.reserve(ng);
            for (int lo = 0, hi = ng - 1; lo <= hi; ++lo, --hi) { mixed.push_back(sig[lo]); if (hi != lo) mixed.push_back(sig[hi]); }
            sig.swap(mixed); }
          group_order.clear();
          for (int q = 0; q < ng; ++q) {
              const int g = sig[q].second;
              if (q & 1) std::reverse(of_group[g].begin(), of_group[g].end());
              group_order.push_back(g);
              for (size_t k = 0; k < of_group[g].size(); ++k) order.push_back(of_group[g][k]);
          } }
        P.n_closings = (int)order.size();
        const int lanes_total = P.nchunks * 32;
        std::vector<unsigned> cfgbits(P.NH, 0);
        P.hel_table.assign((size_t)P.NH * n, 0); P.evalidx.assign((size_t)1 << n, -1);
        for (int h = 0; h < P.NH; ++h) {
            std::vector<int> hv = E.hel_of(kept[h]);
            for (int i = 0; i < n; ++i) { P.hel_table[(size_t)h * n + i] = (int8_t)hv[i]; if (hv[i] > 0) cfgbits[h] |= 1u << i; }
            P.evalidx[cfgbits[h]] = (int16_t)h;
            if (fold_parity) P.evalidx[~cfgbits[h] & ((1u << n) - 1u)] = (int16_t)h;
        }
        // per-lane byte rows (one byte per helicity configuration of every warp): row of a leg set = the variant index the
        // configuration selects in a current over those legs; row of (quark-line pairing, line) = bit 0: the configuration
        // conserves chirality along the closing's quark lines, bit 1: chirality of the closing's own line
        std::map<unsigned, int> vrow; std::map<std::pair<std::vector<std::pair<int, int> >, int>, int> frow;
        auto row_of_mask = [&](unsigned mask) -> int {
            std::map<unsigned, int>::iterator it = vrow.find(mask); if (it != vrow.end()) return it->second;
            const int id = (int)(P.lanerows.size() / lanes_total); vrow[mask] = id;
            for (int lane = 0; lane < lanes_total; ++lane) { const int ch = lane / 32, li = lane % 32, h = ch * P.cpc + li; P.lanerows.push_back((li < P.cpc && h < P.NH) ? (uint8_t)extract(cfgbits[h], mask) : 0); }
            return id;
        };
        auto row_of_flags = [&](std::vector<std::pair<int, int> > pairs, int line_leg) -> int {
            std::sort(pairs.begin(), pairs.end());
            const std::pair<std::vector<std::pair<int, int> >, int> key(pairs, line_leg);
            std::map<std::pair<std::vector<std::pair<int, int> >, int>, int>::iterator it = frow.find(key); if (it != frow.end()) return it->second;
            const int id = (int)(P.lanerows.size() / lanes_total); frow[key] = id;
            for (int lane = 0; lane < lanes_total; ++lane) {
                const int ch = lane / 32, li = lane % 32, h = ch * P.cpc + li; uint8_t b = 0;
                if (li < P.cpc && h < P.NH) {
                    bool valid = true;
                    for (size_t q = 0; q < pairs.size(); ++q) if (chi_of_leg(cfgbits[h], pairs[q].first) != chi_of_leg(cfgbits[h], pairs[q].second)) valid = false;
                    b = (valid ? 1 : 0) | ((line_leg >= 0 && chi_of_leg(cfgbits[h], line_leg) > 0) ? 2 : 0);
                }
                P.lanerows.push_back(b);
            }
            return id;
        };
        // one 16-word record per closing (kind 0-2) or per overflow block of colour updates (kind 3):
        //  [0] kind | reset S << 2 | updates (0..8) << 3 | log2 nv of the 4 operands << 8 (3 bits each)   [1] base a | b << 16   [2] base c | d << 16
        //  [3] variant rows of a, b, c, d (bytes)   [4] flag row | ka << 8 | kb << 16 | kc << 24   [5] coefficient of the amplitude in its group sum
        //  [6..13] colour updates: J element | coefficient index << 16
        const int MAXU = 8;
        double fl_b = 0;
        P.n_entries = 0;
        for (size_t k = 0; k < order.size(); ++k) {
            const int l = order[k]; const Closing& cl = G.closings[l]; const int g = E.group_of[l];
            const bool last = (k + 1 == order.size()) || E.group_of[order[k + 1]] != g;
            int c[4] = {cl.c[0], cl.c[1], cl.c[2], cl.c[3]}, kind = TB_VVV;
            if (cl.kind == AK_GGGG) {      // the three pieces are one function with permuted arguments (eqs. 35a-c)
                kind = TB_GGGG;
                if (cl.piece == 1) { c[1] = cl.c[2]; c[2] = cl.c[3]; c[3] = cl.c[1]; }
                else if (cl.piece == 2) { c[1] = cl.c[3]; c[2] = cl.c[1]; c[3] = cl.c[2]; }
            } else if (cl.kind == AK_IOV) { kind = TB_IOV; c[0] = cl.c[1]; c[1] = cl.c[0]; }      // (psi, psibar, gluon)
            else if (cl.kind != AK_VVV) throw std::runtime_error("closing kind without a table form");
            uint32_t b[4] = {0, 0, 0, 0}, ln[4] = {0, 0, 0, 0}, ks[3] = {0, 0, 0}, rows[4] = {0, 0, 0, 0};
            for (int j = 0; j < 4; ++j) if (c[j] >= 0) { b[j] = (uint32_t)base32[c[j]]; ln[j] = (uint32_t)lognv[c[j]]; rows[j] = (uint32_t)row_of_mask(vm(G.cur[c[j]])); }
            if (kind == TB_VVV) for (int j = 0; j < 3; ++j) { ks[j] = (uint32_t)slot_of(G.cur[c[j]].mask); if (ks[j] > 255) throw std::runtime_error("more than 256 momentum slots"); }
            const uint32_t fr = (uint32_t)row_of_flags(cl.pairs, kind == TB_IOV ? G.cur[c[0]].end_leg : -1);
            const size_t nu = last ? X[g].size() : 0;
            size_t done = 0;
            for (int part = 0; part == 0 || done < nu; ++part) {
                const size_t take = std::min<size_t>(MAXU, nu - done);
                const bool reset = last && done + take == nu;
                uint32_t w[16]; memset(w, 0, sizeof w);
                w[0] = (part == 0 ? (uint32_t)kind : 3u) | ((reset ? 1u : 0u) << 2) | ((uint32_t)take << 3) | (ln[0] << 8) | (ln[1] << 11) | (ln[2] << 14) | (ln[3] << 17);      // updates: 4 bits (0..8)
                w[1] = b[0] | (b[1] << 16); w[2] = b[2] | (b[3] << 16);
                w[3] = rows[0] | (rows[1] << 8) | (rows[2] << 16) | (rows[3] << 24);
                w[4] = fr | (ks[0] << 8) | (ks[1] << 16) | (ks[2] << 24);
                w[5] = coef_of(E.group_lead[l]);
                for (size_t t = 0; t < take; ++t) w[6 + t] = (uint32_t)X[g][done + t].first | (coef_of(X[g][done + t].second) << 16);
                for (int q = 0; q < 16; ++q) P.b_rec.push_back(w[q]);
                P.n_entries++; done += take; fl_b += 4.0 * take;
            }
            P.n_jl += (int)nu;
            fl_b += FlopTable::of_closing(cl.kind) + 4;
        }
        if (P.lanerows.size() / lanes_total > 255) throw std::runtime_error("more than 255 lane rows");
        P.n_rows = (int)(P.lanerows.size() / lanes_total);
        if (P.coef.size() > 65535) throw std::runtime_error("more than 65535 distinct coefficients");
        P.nK = (int)kslot.size();
        P.kmask.assign(P.nK, 0);
        for (std::map<unsigned, int>::iterator it = kslot.begin(); it != kslot.end(); ++it) P.kmask[it->second] = it->first;
        // colour form: per tile of 8 rows, columns from the tile's first row on; then the row products
        double fl_c = 0; for (int t = 0; t < P.Rpad / 8; ++t) fl_c += 32.0 * (P.R - 8 * t); fl_c += 4.0 * P.R;
        P.flops_colour_per_hel = fl_c; P.flops_per_hel = fl_b + fl_c + 1;
        P.flops_phase_a += 34.0 * n + 12.0 * P.nK;          // prologue: polarisation bases, subset momenta, 1/q^2
        P.flops_per_event = P.flops_phase_a + P.NH * P.flops_per_hel;
    }
    std::vector<Frac> cacc;
    std::vector<int> group_order;


    // vertex of a current -> table kind with the operands in the order the device function takes them
    static OpT make_term(int kind, const int* ch, int piece, const Frac& coef) {
        OpT t; t.coef = coef; t.ch[0] = ch[0]; t.ch[1] = ch[1]; t.ch[2] = ch[2];
        switch (kind) {
        case CK_GGG: t.kind = TA_GGG; break;
        case CK_GGGG: t.kind = TA_GGGG;      // jgggx0p: piece 0 (a,b,c), 1 (c,a,b), 2 (b,c,a)
            if (piece == 1) { t.ch[0] = ch[2]; t.ch[1] = ch[0]; t.ch[2] = ch[1]; } else if (piece == 2) { t.ch[0] = ch[1]; t.ch[1] = ch[2]; t.ch[2] = ch[0]; } break;
        case CK_FUSE: t.kind = TA_FUSE; t.ch[0] = ch[1]; t.ch[1] = ch[0]; break;      // graph: (psibar, psi) -> table: (psi, psibar)
        case CK_FG: t.kind = TA_FG; break;
        case CK_BG: t.kind = TA_BG; break;
        default: throw std::runtime_error("current kind without a table form");
        }
        return t;
    }
};

}  // namespace heget
