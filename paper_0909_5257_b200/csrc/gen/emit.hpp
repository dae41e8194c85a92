// heget-b200 process generator, part 3: schedule the current graph and emit one specialised CUDA source per process.
//
// the paper converted MadGraph's FORTRAN into CUDA with a converter program and had to cut big
// programs into pieces for its compiler.  Here the generator owns the whole chain: graph.hpp
// enumerates the currents and closings (eq. 7) and expands their colour (eq. 8); this file
//   1. finds the helicity configurations that are not identically zero (massless quark lines conserve chirality),
//   2. merges colour-basis elements whose amplitudes J are proportional for every phase-space point (their rows of the
//      coefficient matrix c_{alpha l} are proportional) into one, with the exact reduced colour matrix,
//   3. orders the closings so that few currents are alive at a time and every current is computed once,
//   4. counts the floating-point operations of the emitted program, and
//   5. writes the CUDA source: a prologue (helicity-independent part of step a3 and the propagator denominators, once per
//      event, into shared memory) and a rolled loop over helicity configurations whose body is straight-line code of
//      device-library calls (steps a3-a7 of SURVEY.md 8(a)).
#pragma once
#include <cstdio>
#include <cstdarg>
#include <cmath>
#include "graph.hpp"

namespace heget {

struct EmitOptions {
    int block64, block32;      // threads per block
    int jreg_max64, jreg_max32;  // keep J in registers up to this many (reduced) colour elements, else shared memory
    EmitOptions() : block64(128), block32(128), jreg_max64(16), jreg_max32(32) {}
};

// flops of the device-library calls as written in heget_dev.cuh (FMA = 2, complex multiply = 6, complex add = 2)
struct FlopTable {
    static int of_current(int kind) {
        switch (kind) { case CK_GGG: return 157; case CK_GGGG: return 65; case CK_FUSE: return 42; case CK_FG: case CK_BG: return 74; case CK_OPEN3: return 157; case CK_OPEN4: return 65; default: return 0; }
    }
    static int of_closing(int kind) { switch (kind) { case AK_VVV: return 168; case AK_GGGG: return 70; case AK_DOT: return 30; default: return 58; } }
};

// Closings that differ in ONE of their currents share the rest of the vertex: V3(a,b,c) = open3(a,b) . c (cyclic in a,b,c) and
// W_piece(a,b,c,d) = open4(a,b,c;piece) . d, where open* is the off-shell current of that vertex without its propagator
// (checked numerically against vvvxxx / ggggxxp).  A 3-leg sub-tree comes in several colour pieces, all closing on the same
// partner currents: the open vertex is built once (150 flops) and every piece costs a 4-vector product (30 flops) instead of a
// full vvvxxx (168).  The open vertices are ordinary nodes of the current graph, so the scheduler places them like any current.
static inline void share_closings(Graph& G) {
    typedef std::vector<int> Key;
    std::map<Key, int> count;
    for (size_t l = 0; l < G.closings.size(); ++l) {
        const Closing& cl = G.closings[l];
        if (cl.kind == AK_VVV) for (int r = 0; r < 3; ++r) { Key k; k.push_back(0); k.push_back(cl.c[r]); k.push_back(cl.c[(r + 1) % 3]); count[k]++; }
        else if (cl.kind == AK_GGGG) { Key k; k.push_back(1); k.push_back(cl.c[0]); k.push_back(cl.c[1]); k.push_back(cl.c[2]); k.push_back(cl.piece); count[k]++; }
    }
    std::map<Key, int> made;
    for (size_t l = 0; l < G.closings.size(); ++l) {
        Closing& cl = G.closings[l];
        Key best; int bestn = 1, rest = -1;
        if (cl.kind == AK_VVV) {
            for (int r = 0; r < 3; ++r) { Key k; k.push_back(0); k.push_back(cl.c[r]); k.push_back(cl.c[(r + 1) % 3]); if (count[k] > bestn) { bestn = count[k]; best = k; rest = cl.c[(r + 2) % 3]; } }
        } else if (cl.kind == AK_GGGG) {
            Key k; k.push_back(1); k.push_back(cl.c[0]); k.push_back(cl.c[1]); k.push_back(cl.c[2]); k.push_back(cl.piece);
            if (count[k] > bestn) { bestn = count[k]; best = k; rest = cl.c[3]; }
        }
        if (rest < 0) continue;
        if (!made.count(best)) {
            Cur W; W.id = (int)G.cur.size(); W.ptype = PT_G; W.end_leg = -1; W.leg = -1; W.piece = best[0] ? best[4] : 0;
            W.kind = best[0] ? CK_OPEN4 : CK_OPEN3;
            W.ch[0] = best[1]; W.ch[1] = best[2]; W.ch[2] = best[0] ? best[3] : -1;
            W.mask = 0; W.varmask = 0; W.size = 0;
            for (int j = 0; j < 3; ++j) if (W.ch[j] >= 0) {
                const Cur& c = G.cur[W.ch[j]];
                W.mask |= c.mask; W.varmask |= c.varmask; W.size += c.size;
                for (size_t q = 0; q < c.pairs.size(); ++q) W.pairs.push_back(c.pairs[q]);
            }
            std::sort(W.pairs.begin(), W.pairs.end());
            made[best] = W.id; G.cur.push_back(W);
        }
        cl.kind = AK_DOT; cl.c[0] = made[best]; cl.c[1] = rest; cl.c[2] = cl.c[3] = -1;
    }
}

struct Emitter {
    const Graph& G;
    std::string tag;
    EmitOptions opt;
    int n, ng, nq;
    std::vector<int> gluon_legs, quark_legs;
    // helicity configurations
    std::vector<std::vector<int> > qcfg;          // valid quark-helicity assignments (one entry per quark leg, +-1)
    std::vector<unsigned> qact;                   // per valid assignment: bit g set = guard g is satisfied
    std::map<std::vector<std::pair<int, int> >, int> guard_of;
    int NH;
    // reduced colour basis
    std::vector<int> class_of; std::vector<Frac> scale_of; int NJ;
    std::vector<Frac> Cred;
    // event-cache slots
    std::vector<int> leg_slot; std::map<unsigned, int> kslot, islot; int nslots;
    // schedule
    struct Op { bool closing; int id; };
    std::vector<Op> ops;
    std::vector<int> last_use;                    // per current: index of the last op reading it
    int max_live;
    double flops_hel, flops_colour, flops_prologue;
    std::string out;

    Emitter(const Graph& g, const std::string& t, const EmitOptions& o) : G(g), tag(t), opt(o) {}

    void pf(const char* fmt, ...) {
        char buf[4096]; va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap); out += buf;
    }
    static int chi_of(const Leg& L, int h) { return -h * (L.anti ? -1 : 1); }

    // ---- 1. helicity configurations ------------------------------------------------------------------------------
    void analyse_helicities() {
        n = G.P.n; gluon_legs.clear(); quark_legs.clear();
        for (int i = 0; i < n; ++i) (G.P.legs[i].type == LEG_G ? gluon_legs : quark_legs).push_back(i);
        ng = (int)gluon_legs.size(); nq = (int)quark_legs.size();
        // guards = distinct sets of completed quark lines
        for (size_t c = 0; c < G.cur.size(); ++c) add_guard(G.cur[c].pairs);
        for (size_t l = 0; l < G.closings.size(); ++l) add_guard(G.closings[l].pairs);
        if (guard_of.size() > 31) throw std::runtime_error("too many chirality guards");
        for (int bits = 0; bits < (1 << nq); ++bits) {
            std::vector<int> hel(nq), chi(n, 0);
            for (int j = 0; j < nq; ++j) { hel[j] = ((bits >> j) & 1) ? +1 : -1; chi[quark_legs[j]] = chi_of(G.P.legs[quark_legs[j]], hel[j]); }
            unsigned act = 0;
            for (std::map<std::vector<std::pair<int, int> >, int>::iterator it = guard_of.begin(); it != guard_of.end(); ++it) {
                bool ok = true;
                for (size_t k = 0; k < it->first.size(); ++k) if (chi[it->first[k].first] != chi[it->first[k].second]) ok = false;
                if (ok) act |= 1u << it->second;
            }
            bool any = false;
            for (size_t l = 0; l < G.closings.size(); ++l) if (act & (1u << guard(G.closings[l].pairs))) { any = true; break; }
            if (any) { qcfg.push_back(hel); qact.push_back(act); }
        }
        NH = (int)qcfg.size() << ng;
    }
    void add_guard(std::vector<std::pair<int, int> > p) { std::sort(p.begin(), p.end()); if (!guard_of.count(p)) { int id = (int)guard_of.size(); guard_of[p] = id; } }
    int guard(std::vector<std::pair<int, int> > p) const { std::sort(p.begin(), p.end()); return guard_of.find(p)->second; }
    bool guard_trivial(int g) const { for (size_t i = 0; i < qact.size(); ++i) if (!(qact[i] & (1u << g))) return false; return true; }

    // ---- 2. reduced colour basis -----------------------------------------------------------------------------------
    void reduce_colour() {
        const int m = (int)G.basis.size();
        std::vector<std::vector<std::pair<int, Frac> > > row(m);
        for (size_t l = 0; l < G.closings.size(); ++l)
            for (size_t t = 0; t < G.closings[l].coef.size(); ++t) row[G.closings[l].coef[t].first].push_back(std::make_pair((int)l, G.closings[l].coef[t].second));
        std::map<std::vector<std::pair<int, std::pair<long long, long long> > >, int> seen;
        class_of.assign(m, -1); scale_of.assign(m, Frac(0)); NJ = 0;
        for (int a = 0; a < m; ++a) {
            if (row[a].empty()) throw std::runtime_error("colour basis element without diagram");
            const Frac lead = row[a][0].second, inv(lead.d, lead.n);
            std::vector<std::pair<int, std::pair<long long, long long> > > key;
            for (size_t t = 0; t < row[a].size(); ++t) { Frac r = row[a][t].second * inv; key.push_back(std::make_pair(row[a][t].first, std::make_pair(r.n, r.d))); }
            std::map<std::vector<std::pair<int, std::pair<long long, long long> > >, int>::iterator it = seen.find(key);
            if (it == seen.end()) { seen[key] = NJ; class_of[a] = NJ++; rep.push_back(a); scale_of[a] = Frac(1); }
            else { class_of[a] = it->second; const Frac l0 = row[rep[it->second]][0].second; scale_of[a] = lead * Frac(l0.d, l0.n); }
        }
        Cred.assign((size_t)NJ * NJ, Frac(0));
        for (int a = 0; a < m; ++a) for (int b = 0; b < m; ++b) {
            Frac& c = Cred[(size_t)class_of[a] * NJ + class_of[b]];
            c = c + scale_of[a] * scale_of[b] * G.C[(size_t)a * m + b];
        }
    }
    std::vector<int> rep;

    // ---- 3. schedule -----------------------------------------------------------------------------------------------
    int cost_missing(int c, std::vector<char>& done, std::vector<int>& stamp, int mark) const {
        if (done[c] || stamp[c] == mark) return 0;
        stamp[c] = mark;
        const Cur& C = G.cur[c];
        if (C.kind == CK_LEAF) return 0;
        int s = 1;
        for (int j = 0; j < 3; ++j) if (C.ch[j] >= 0) s += cost_missing(C.ch[j], done, stamp, mark);
        return s;
    }
    void need(int c, std::vector<char>& done) {
        if (done[c]) return;
        const Cur& C = G.cur[c];
        for (int j = 0; j < 3; ++j) if (C.ch[j] >= 0) need(C.ch[j], done);
        done[c] = 1;
        if (C.kind != CK_LEAF) { Op o; o.closing = false; o.id = c; ops.push_back(o); }
    }
    // transitive set of not-yet-computed currents under c (post-order), without marking them done
    void missing(int c, const std::vector<char>& done, std::vector<int>& stamp, int mark, std::vector<int>& out) const {
        if (done[c] || stamp[c] == mark) return;
        stamp[c] = mark;
        const Cur& C = G.cur[c];
        if (C.kind == CK_LEAF) return;
        for (int j = 0; j < 3; ++j) if (C.ch[j] >= 0) missing(C.ch[j], done, stamp, mark, out);
        out.push_back(c);
    }
    void schedule() {
        const int nc = (int)G.cur.size(), nl = (int)G.closings.size();
        std::vector<char> done(nc, 0);
        std::vector<int> stamp(nc, -1);
        int mark = 0;
        // uses[c] = ops (currents that will certainly be needed, closings) still to read current c
        std::vector<char> needed(nc, 0);
        { std::vector<int> st; for (int l = 0; l < nl; ++l) for (int j = 0; j < 4; ++j) if (G.closings[l].c[j] >= 0) st.push_back(G.closings[l].c[j]);
          while (!st.empty()) { int c = st.back(); st.pop_back(); if (needed[c]) continue; needed[c] = 1; for (int j = 0; j < 3; ++j) if (G.cur[c].ch[j] >= 0) st.push_back(G.cur[c].ch[j]); } }
        std::vector<int> uses(nc, 0);
        for (int c = 0; c < nc; ++c) if (needed[c]) for (int j = 0; j < 3; ++j) if (G.cur[c].ch[j] >= 0) uses[G.cur[c].ch[j]]++;
        for (int l = 0; l < nl; ++l) for (int j = 0; j < 4; ++j) if (G.closings[l].c[j] >= 0) uses[G.closings[l].c[j]]++;
        // Greedy for a small peak of simultaneously live currents (each is 8 or 16 registers): take the closing whose
        // execution changes the number of live currents the least (new currents that stay alive minus currents that die),
        // then the one that needs the fewest new currents, then generator order.
        std::vector<int> pending; for (int l = 0; l < nl; ++l) pending.push_back(l);
        std::vector<int> tmp(nc, 0), miss;
        while (!pending.empty()) {
            int best = -1; long bestscore = 1L << 40; size_t bestpos = 0;
            for (size_t k = 0; k < pending.size(); ++k) {
                const Closing& cl = G.closings[pending[k]];
                ++mark; miss.clear();
                for (int j = 0; j < 4; ++j) if (cl.c[j] >= 0) missing(cl.c[j], done, stamp, mark, miss);
                // simulate the use counts
                std::vector<int> touched;
                for (size_t m = 0; m < miss.size(); ++m) for (int j = 0; j < 3; ++j) { const int ch = G.cur[miss[m]].ch[j]; if (ch >= 0) { if (!tmp[ch]) touched.push_back(ch); tmp[ch]++; } }
                for (int j = 0; j < 4; ++j) if (cl.c[j] >= 0) { const int ch = cl.c[j]; if (!tmp[ch]) touched.push_back(ch); tmp[ch]++; }
                int born = 0, dying = 0, closest = 255;
                for (size_t m = 0; m < miss.size(); ++m) if (uses[miss[m]] - tmp[miss[m]] > 0 && G.cur[miss[m]].kind != CK_OPEN3 && G.cur[miss[m]].kind != CK_OPEN4) ++born;   // new and still needed afterwards (open vertices are short-lived helpers of the currents already alive: not charged)
                for (size_t q = 0; q < touched.size(); ++q) {
                    const int ch = touched[q];
                    if (G.cur[ch].kind == CK_LEAF || !done[ch]) continue;
                    const int left = uses[ch] - tmp[ch];
                    if (left == 0) ++dying;
                    // "finish what was started": among equal changes prefer the closing that brings a big live current nearest to its death
                    const int key = left * 4 - G.cur[ch].size; if (key < closest) closest = key < 0 ? 0 : key;
                }
                for (size_t q = 0; q < touched.size(); ++q) tmp[touched[q]] = 0;
                const long score = (long)(born - dying) * (1L << 20) + (long)closest * 256 + (long)miss.size();
                if (score < bestscore) { bestscore = score; best = pending[k]; bestpos = k; }
            }
            const Closing& cl = G.closings[best];
            ++mark; miss.clear();
            for (int j = 0; j < 4; ++j) if (cl.c[j] >= 0) missing(cl.c[j], done, stamp, mark, miss);
            for (size_t m = 0; m < miss.size(); ++m) {
                done[miss[m]] = 1; Op o; o.closing = false; o.id = miss[m]; ops.push_back(o);
                for (int j = 0; j < 3; ++j) if (G.cur[miss[m]].ch[j] >= 0) uses[G.cur[miss[m]].ch[j]]--;
            }
            for (int j = 0; j < 4; ++j) if (cl.c[j] >= 0) uses[cl.c[j]]--;
            Op o; o.closing = true; o.id = best; ops.push_back(o);
            pending.erase(pending.begin() + bestpos);
        }
        const int ncd = nc; (void)ncd;
        // liveness
        last_use.assign(nc, -1);
        for (size_t k = 0; k < ops.size(); ++k) {
            if (ops[k].closing) { const Closing& cl = G.closings[ops[k].id]; for (int j = 0; j < 4; ++j) if (cl.c[j] >= 0) last_use[cl.c[j]] = (int)k; }
            else { const Cur& C = G.cur[ops[k].id]; for (int j = 0; j < 3; ++j) if (C.ch[j] >= 0) last_use[C.ch[j]] = (int)k; }
        }
        max_live = 0; int live = 0;
        std::vector<int> dies(ops.size() + 1, 0);
        for (int c = 0; c < nc; ++c) if (G.cur[c].kind != CK_LEAF && last_use[c] >= 0) dies[last_use[c]]++;
        for (size_t k = 0; k < ops.size(); ++k) { if (!ops[k].closing) ++live; if (live > max_live) max_live = live; live -= dies[k]; }
    }

    // ---- event-cache slots -----------------------------------------------------------------------------------------
    void assign_slots() {
        nslots = 0; leg_slot.assign(n, -1);
        for (int i = 0; i < n; ++i) { leg_slot[i] = nslots; nslots += (G.P.legs[i].type == LEG_G) ? 6 : 3; }
        for (size_t c = 0; c < G.cur.size(); ++c) {
            const unsigned m = G.cur[c].mask;
            if (!kslot.count(m)) { kslot[m] = nslots; nslots += 4; if (G.cur[c].size >= 2) { islot[m] = nslots; nslots += 1; } }
        }
    }
#include "emit_body.inc"
};
}  // namespace heget
