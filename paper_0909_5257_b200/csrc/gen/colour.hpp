// heget-b200 process generator, part 1: exact SU(3) colour algebra on index strings.
//
// PAPER.md:81-91 (eqs. 8-10): every diagram's colour factor is expanded on a colour basis T_alpha made of
// products/traces of fundamental generators, and |M|^2 needs the matrix C_ab = sum_colours T_a (T_b)^*.
// Here both are obtained SYMBOLICALLY and EXACTLY (rational arithmetic, N = 3):
//   * a colour object is a linear combination of products of "strings": an open string
//     (T^{s1} ... T^{sk})_{head tail} runs along a quark line (head = colour index of the line's out-end,
//     tail = of its in-end), a closed string is a trace Tr(T^{s1} ... T^{sk});
//   * symbols are external gluon legs (>= 0), the open adjoint index of an off-shell gluon (MARK), and
//     summed dummy indices (< MARK);
//   * vertices are written with generators only:  i f^{abc} = 2 Tr(T^a T^b T^c) - 2 Tr(T^b T^a T^c)
//     (colour factor of eq. 27/30), -T^a_{ij} for the quark-gluon vertex (eq. 22);
//   * a summed index is removed with the Fierz identity
//         T^a_{ij} T^a_{kl} = 1/2 ( delta_il delta_kj - 1/N delta_ij delta_kl ).
// Normalisation: T^a = lambda^a/2, Tr(T^a T^b) = delta^{ab}/2.
// This file is part of the PRODUCT (host side of the generator).  It shares nothing with oracle/.
#pragma once
#include <vector>
#include <map>
#include <algorithm>
#include <stdexcept>
#include <cstdlib>
#include <string>

namespace heget {

static inline long long gcd_ll(long long a, long long b) { a = std::llabs(a); b = std::llabs(b); while (b) { long long t = a % b; a = b; b = t; } return a ? a : 1; }

struct Frac {
    long long n, d;
    Frac(long long n_ = 0, long long d_ = 1) : n(n_), d(d_) { norm(); }
    void norm() { if (d < 0) { n = -n; d = -d; } long long g = gcd_ll(n, d); n /= g; d /= g; if (n == 0) d = 1; }
    Frac operator*(const Frac& o) const { long long g1 = gcd_ll(n, o.d), g2 = gcd_ll(o.n, d); return Frac((n / g1) * (o.n / g2), (d / g2) * (o.d / g1)); }
    Frac operator+(const Frac& o) const { long long g = gcd_ll(d, o.d); return Frac(n * (o.d / g) + o.n * (d / g), (d / g) * o.d); }
    Frac operator-() const { return Frac(-n, d); }
    Frac operator-(const Frac& o) const { return *this + (-o); }
    bool zero() const { return n == 0; }
    bool operator==(const Frac& o) const { return n == o.n && d == o.d; }
    bool operator<(const Frac& o) const { return (__int128)n * o.d < (__int128)o.n * d; }
    double value() const { return (double)n / (double)d; }
};

typedef int Sym;
static const Sym MARK = -1;        // open adjoint index of an off-shell gluon
static const Sym BRIDGE = -2;      // the one gluon exchanged between two quark lines, kept summed ("paper" basis)
static const Sym BRIDGE2 = -3;     // same, of the conjugated element when building the colour matrix
static const int OPEN_END = -1000; // open fundamental index of an off-shell quark
static const int NC = 3;

struct CString {
    bool closed;
    int head, tail;                // open strings: external quark leg carrying the index, or OPEN_END
    std::vector<Sym> s;
    bool operator<(const CString& o) const {
        if (closed != o.closed) return closed < o.closed;
        if (head != o.head) return head < o.head;
        if (tail != o.tail) return tail < o.tail;
        return s < o.s;
    }
    bool operator==(const CString& o) const { return closed == o.closed && head == o.head && tail == o.tail && s == o.s; }
};

struct CTerm {
    std::vector<CString> strs;
    bool operator<(const CTerm& o) const { return strs < o.strs; }
    bool operator==(const CTerm& o) const { return strs == o.strs; }
    void canon() {
        for (size_t i = 0; i < strs.size(); ++i) if (strs[i].closed && !strs[i].s.empty()) {
            std::vector<Sym>& v = strs[i].s;
            // rotate the smallest NON-NEGATIVE symbol to the front (externals are unique); dummies/MARK sort after
            size_t best = 0; bool have = false;
            for (size_t k = 0; k < v.size(); ++k) {
                if (v[k] < 0) continue;
                if (!have || v[k] < v[best]) { best = k; have = true; }
            }
            if (!have) { for (size_t k = 1; k < v.size(); ++k) if (v[k] > v[best]) best = k; }   // MARK (=-1) first
            std::rotate(v.begin(), v.begin() + best, v.end());
        }
        std::sort(strs.begin(), strs.end());
    }
};

typedef std::map<CTerm, Frac> CExpr;

static inline void add_term(CExpr& e, CTerm t, const Frac& c) {
    if (c.zero()) return;
    t.canon();
    CExpr::iterator it = e.find(t);
    if (it == e.end()) e[t] = c;
    else { it->second = it->second + c; if (it->second.zero()) e.erase(it); }
}

static inline CExpr scaled(const CExpr& e, const Frac& f) { CExpr r; for (CExpr::const_iterator it = e.begin(); it != e.end(); ++it) r[it->first] = it->second * f; return r; }
static inline CExpr sum(const CExpr& a, const CExpr& b) { CExpr r = a; for (CExpr::const_iterator it = b.begin(); it != b.end(); ++it) add_term(r, it->first, it->second); return r; }

static inline CExpr product(const CExpr& a, const CExpr& b) {
    CExpr r;
    for (CExpr::const_iterator i = a.begin(); i != a.end(); ++i) for (CExpr::const_iterator j = b.begin(); j != b.end(); ++j) {
        CTerm t = i->first; t.strs.insert(t.strs.end(), j->first.strs.begin(), j->first.strs.end());
        add_term(r, t, i->second * j->second);
    }
    return r;
}

static inline CExpr renamed(const CExpr& e, Sym from, Sym to) {
    CExpr r;
    for (CExpr::const_iterator it = e.begin(); it != e.end(); ++it) {
        CTerm t = it->first;
        for (size_t i = 0; i < t.strs.size(); ++i) for (size_t k = 0; k < t.strs[i].s.size(); ++k) if (t.strs[i].s[k] == from) t.strs[i].s[k] = to;
        add_term(r, t, it->second);
    }
    return r;
}

static inline CExpr trace_expr(const std::vector<Sym>& v, const Frac& c) {
    CString s; s.closed = true; s.head = s.tail = 0; s.s = v;
    CTerm t; t.strs.push_back(s);
    CExpr e; add_term(e, t, c); return e;
}

// a closed string with 0 symbols is Tr(1) = N, with 1 symbol Tr(T^a) = 0.  Returns false if the term dies.
static inline bool absorb_trivial(CTerm& t, Frac& c) {
    for (size_t i = 0; i < t.strs.size();) {
        if (t.strs[i].closed && t.strs[i].s.size() <= 1) {
            if (t.strs[i].s.size() == 1) return false;
            c = c * Frac(NC); t.strs.erase(t.strs.begin() + i);
        } else ++i;
    }
    return true;
}

// Remove the summed index d (appearing exactly twice per term) by the Fierz identity.
// keep_bridge: if the two occurrences sit on two different OPEN strings, keep the sum and rename d -> BRIDGE.
static inline CExpr contract(const CExpr& e, Sym d, bool keep_bridge) {
    CExpr r;
    for (CExpr::const_iterator it = e.begin(); it != e.end(); ++it) {
        const CTerm& t = it->first;
        int s1 = -1, p1 = -1, s2 = -1, p2 = -1;
        for (size_t i = 0; i < t.strs.size(); ++i) for (size_t k = 0; k < t.strs[i].s.size(); ++k) if (t.strs[i].s[k] == d) {
            if (s1 < 0) { s1 = (int)i; p1 = (int)k; } else { s2 = (int)i; p2 = (int)k; }
        }
        if (s1 < 0) { add_term(r, t, it->second); continue; }
        if (s2 < 0) throw std::runtime_error("colour: summed index appears once");
        CTerm rest; for (size_t i = 0; i < t.strs.size(); ++i) if ((int)i != s1 && (int)i != s2) rest.strs.push_back(t.strs[i]);
        const Frac half(1, 2), mhalfN(-1, 2 * NC);
        if (s1 == s2) {
            const CString& S = t.strs[s1];
            std::vector<Sym> A(S.s.begin(), S.s.begin() + p1), B(S.s.begin() + p1 + 1, S.s.begin() + p2), Cc(S.s.begin() + p2 + 1, S.s.end());
            // A d B d C  ->  1/2 (A C) Tr(B) - 1/(2N) (A B C)
            CString outer = S; outer.s = A; outer.s.insert(outer.s.end(), Cc.begin(), Cc.end());
            CString inner; inner.closed = true; inner.head = inner.tail = 0; inner.s = B;
            { CTerm n = rest; n.strs.push_back(outer); n.strs.push_back(inner); Frac c = it->second * half; if (absorb_trivial(n, c)) add_term(r, n, c); }
            CString all = S; all.s = A; all.s.insert(all.s.end(), B.begin(), B.end()); all.s.insert(all.s.end(), Cc.begin(), Cc.end());
            { CTerm n = rest; n.strs.push_back(all); Frac c = it->second * mhalfN; if (absorb_trivial(n, c)) add_term(r, n, c); }
        } else {
            const CString& S = t.strs[s1]; const CString& U = t.strs[s2];
            if (keep_bridge && !S.closed && !U.closed) {
                CTerm n = t; n.strs[s1].s[p1] = BRIDGE; n.strs[s2].s[p2] = BRIDGE; add_term(r, n, it->second); continue;
            }
            std::vector<Sym> A(S.s.begin(), S.s.begin() + p1), B(S.s.begin() + p1 + 1, S.s.end());
            std::vector<Sym> Cc(U.s.begin(), U.s.begin() + p2), D(U.s.begin() + p2 + 1, U.s.end());
            // (A d B)(C d D) -> 1/2 (A D)(C B) - 1/(2N) (A B)(C D)
            {
                CTerm n = rest;
                if (S.closed && U.closed) { CString x; x.closed = true; x.head = x.tail = 0; x.s = A; x.s.insert(x.s.end(), D.begin(), D.end()); x.s.insert(x.s.end(), Cc.begin(), Cc.end()); x.s.insert(x.s.end(), B.begin(), B.end()); n.strs.push_back(x); }
                else if (S.closed) { CString x = U; x.s = Cc; x.s.insert(x.s.end(), B.begin(), B.end()); x.s.insert(x.s.end(), A.begin(), A.end()); x.s.insert(x.s.end(), D.begin(), D.end()); n.strs.push_back(x); }
                else if (U.closed) { CString x = S; x.s = A; x.s.insert(x.s.end(), D.begin(), D.end()); x.s.insert(x.s.end(), Cc.begin(), Cc.end()); x.s.insert(x.s.end(), B.begin(), B.end()); n.strs.push_back(x); }
                else {
                    CString x; x.closed = false; x.head = S.head; x.tail = U.tail; x.s = A; x.s.insert(x.s.end(), D.begin(), D.end());
                    CString y; y.closed = false; y.head = U.head; y.tail = S.tail; y.s = Cc; y.s.insert(y.s.end(), B.begin(), B.end());
                    n.strs.push_back(x); n.strs.push_back(y);
                }
                Frac c = it->second * half; if (absorb_trivial(n, c)) add_term(r, n, c);
            }
            {
                CTerm n = rest;
                CString x = S; x.s = A; x.s.insert(x.s.end(), B.begin(), B.end());
                CString y = U; y.s = Cc; y.s.insert(y.s.end(), D.begin(), D.end());
                n.strs.push_back(x); n.strs.push_back(y);
                Frac c = it->second * mhalfN; if (absorb_trivial(n, c)) add_term(r, n, c);
            }
        }
    }
    return r;
}

struct ColourAlgebra {
    bool keep_bridge;
    int next_dummy;
    ColourAlgebra() : keep_bridge(false), next_dummy(-10) {}
    Sym fresh() { return next_dummy--; }

    // ---- leaves --------------------------------------------------------------------------
    CExpr leaf_gluon(int leg) { std::vector<Sym> v; v.push_back(MARK); v.push_back(leg); return trace_expr(v, Frac(2)); }   // delta^{MARK leg}
    CExpr leaf_psi(int leg) { CString s; s.closed = false; s.head = OPEN_END; s.tail = leg; CTerm t; t.strs.push_back(s); CExpr e; add_term(e, t, Frac(1)); return e; }
    CExpr leaf_psibar(int leg) { CString s; s.closed = false; s.head = leg; s.tail = OPEN_END; CTerm t; t.strs.push_back(s); CExpr e; add_term(e, t, Frac(1)); return e; }

    // ---- off-shell currents ----------------------------------------------------------------
    // z_c = i f^{abc} x_a y_b                                             (eq. 30)
    CExpr join3(const CExpr& X, const CExpr& Y) {
        Sym a = fresh(), b = fresh();
        std::vector<Sym> v1, v2; v1.push_back(a); v1.push_back(b); v1.push_back(MARK); v2.push_back(b); v2.push_back(a); v2.push_back(MARK);
        CExpr V = sum(trace_expr(v1, Frac(2)), trace_expr(v2, Frac(-2)));
        CExpr e = product(product(renamed(X, MARK, a), renamed(Y, MARK, b)), V);
        e = contract(e, a, keep_bridge);
        return contract(e, b, keep_bridge);
    }
    // the three colour structures of the four-gluon vertex (eq. 40), open index d:
    //   piece 0: f^{abe}f^{cde}   piece 1: f^{ace}f^{dbe}   piece 2: f^{ade}f^{bce}
    // (i f^{abe})(i f^{ecd}) = -f^{abe}f^{cde};  (i f^{ace})(i f^{ebd}) = +f^{ace}f^{dbe};  (i f^{bce})(i f^{aed}) = +f^{ade}f^{bce}
    CExpr join4(const CExpr& X, const CExpr& Y, const CExpr& Z, int piece) {
        if (piece == 0) return scaled(join3(join3(X, Y), Z), Frac(-1));
        if (piece == 1) return join3(join3(X, Z), Y);
        return join3(X, join3(Y, Z));
    }
    // quark + gluon -> quark, colour factor -T^a_{ij} (eq. 22): the generator goes on the open end
    CExpr attach(const CExpr& Q, const CExpr& G, bool psi) {
        Sym a = fresh();
        CExpr p = product(Q, renamed(G, MARK, a));
        CExpr q;
        for (CExpr::const_iterator it = p.begin(); it != p.end(); ++it) {
            CTerm t = it->first; bool done = false;
            for (size_t i = 0; i < t.strs.size() && !done; ++i) if (!t.strs[i].closed) {
                if (psi && t.strs[i].head == OPEN_END) { t.strs[i].s.insert(t.strs[i].s.begin(), a); done = true; }
                else if (!psi && t.strs[i].tail == OPEN_END) { t.strs[i].s.push_back(a); done = true; }
            }
            if (!done) throw std::runtime_error("colour: no open quark end");
            add_term(q, t, -it->second);
        }
        return contract(q, a, keep_bridge);
    }
    // psibar + psi -> gluon, colour factor -T^MARK_{ij}
    CExpr fuse(const CExpr& B, const CExpr& F, Sym mid) {
        CExpr r;
        for (CExpr::const_iterator i = B.begin(); i != B.end(); ++i) for (CExpr::const_iterator j = F.begin(); j != F.end(); ++j) {
            CTerm t; CString m; m.closed = false; bool hb = false, hf = false;
            for (size_t k = 0; k < i->first.strs.size(); ++k) { const CString& s = i->first.strs[k]; if (!s.closed && s.tail == OPEN_END) { m.head = s.head; m.s = s.s; hb = true; } else t.strs.push_back(s); }
            m.s.push_back(mid);
            for (size_t k = 0; k < j->first.strs.size(); ++k) { const CString& s = j->first.strs[k]; if (!s.closed && s.head == OPEN_END) { m.tail = s.tail; m.s.insert(m.s.end(), s.s.begin(), s.s.end()); hf = true; } else t.strs.push_back(s); }
            if (!hb || !hf) throw std::runtime_error("colour: fuse needs psibar and psi");
            t.strs.push_back(m);
            add_term(r, t, -(i->second * j->second));
        }
        return r;
    }
    CExpr fuse_gluon(const CExpr& B, const CExpr& F) { return fuse(B, F, MARK); }

    // ---- closings (amplitudes): all indices summed ----------------------------------------------
    CExpr dot(const CExpr& X, const CExpr& Y) { Sym c = fresh(); return contract(product(renamed(X, MARK, c), renamed(Y, MARK, c)), c, keep_bridge); }
    CExpr amp_vvv(const CExpr& X, const CExpr& Y, const CExpr& Z) { return dot(join3(X, Y), Z); }
    CExpr amp_gggg(const CExpr& X, const CExpr& Y, const CExpr& Z, const CExpr& W, int piece) { return dot(join4(X, Y, Z, piece), W); }
    CExpr amp_iov(const CExpr& B, const CExpr& F, const CExpr& G) { Sym a = fresh(); return contract(product(fuse(B, F, a), renamed(G, MARK, a)), a, keep_bridge); }

    // ---- colour matrix element  sum_colours  t1 * conj(t2)  ---------------------------------------
    // conj of a string = reversed string with head/tail exchanged (T^a hermitian)
    Frac overlap(const CTerm& t1, const CTerm& t2, const std::vector<int>& gluon_legs) {
        CTerm t = t1;
        for (size_t i = 0; i < t2.strs.size(); ++i) {
            CString s = t2.strs[i]; std::reverse(s.s.begin(), s.s.end());
            for (size_t k = 0; k < s.s.size(); ++k) if (s.s[k] == BRIDGE) s.s[k] = BRIDGE2;
            if (!s.closed) std::swap(s.head, s.tail);
            t.strs.push_back(s);
        }
        // join open strings through their shared external quark indices until only traces remain
        for (;;) {
            int a = -1; for (size_t i = 0; i < t.strs.size(); ++i) if (!t.strs[i].closed) { a = (int)i; break; }
            if (a < 0) break;
            CString S = t.strs[a]; t.strs.erase(t.strs.begin() + a);
            while (S.head != S.tail || S.closed) {
                int b = -1; for (size_t i = 0; i < t.strs.size(); ++i) if (!t.strs[i].closed && t.strs[i].head == S.tail) { b = (int)i; break; }
                if (b < 0) throw std::runtime_error("colour: unmatched quark index");
                S.s.insert(S.s.end(), t.strs[b].s.begin(), t.strs[b].s.end()); S.tail = t.strs[b].tail; t.strs.erase(t.strs.begin() + b);
                if (S.head == S.tail) break;
            }
            S.closed = true; S.head = S.tail = 0; t.strs.push_back(S);
        }
        CExpr e; Frac one(1);
        if (!absorb_trivial(t, one)) return Frac(0);
        add_term(e, t, one);
        std::vector<Sym> todo(gluon_legs.begin(), gluon_legs.end()); todo.push_back(BRIDGE); todo.push_back(BRIDGE2);
        for (size_t k = 0; k < todo.size(); ++k) e = contract(e, todo[k], false);
        Frac r(0);
        for (CExpr::const_iterator it = e.begin(); it != e.end(); ++it) { if (!it->first.strs.empty()) throw std::runtime_error("colour: overlap not a number"); r = r + it->second; }
        return r;
    }
};

static inline std::string term_to_string(const CTerm& t) {
    std::string o;
    for (size_t i = 0; i < t.strs.size(); ++i) {
        const CString& s = t.strs[i];
        o += s.closed ? "Tr(" : "(";
        for (size_t k = 0; k < s.s.size(); ++k) { if (k) o += " "; o += s.s[k] == BRIDGE ? "e" : (s.s[k] == MARK ? "*" : std::to_string(s.s[k])); }
        o += ")";
        if (!s.closed) o += "_{" + std::to_string(s.head) + "," + std::to_string(s.tail) + "}";
    }
    return o;
}
}  // namespace heget
