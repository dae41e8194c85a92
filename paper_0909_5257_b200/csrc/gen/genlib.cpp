// In-process entry to the process generator (step a0), used by
// heget_process_create when no pre-built plug-in exists for a process.  Same work as the hegetgen command line.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <fstream>
#include "emit.hpp"
#include "tab.hpp"

using namespace heget;

// returns 0 = source written, 1 = malformed process, 2 = valid syntax but unsupported / too large, 3 = I/O or internal error
extern "C" int heget_generate_source(const char* tag, const char* process, const char* out_path, char* msg, int msglen) {
    try {
        Process P;
        try { P = parse_process(process); }
        catch (std::invalid_argument& e) { snprintf(msg, msglen, "%s", e.what()); return 2; }
        catch (std::exception& e) { snprintf(msg, msglen, "%s", e.what()); return 1; }
        if (P.n > 7) { snprintf(msg, msglen, "process with %d external legs is too large to build", P.n); return 2; }
        int q = 0; for (int i = 0; i < P.n; ++i) q += P.legs[i].type != LEG_G;
        Graph G, GP; const Graph* paper = 0;
        try {
            G.build(P, false);
            if (q == 4) { GP.build(P, true); paper = &GP; }
        } catch (std::exception& e) { snprintf(msg, msglen, "%s", e.what()); return 2; }
        if (G.closings.empty()) { snprintf(msg, msglen, "process has no tree-level QCD diagram"); return 2; }
        EmitOptions opt;
        Emitter E(G, tag, opt);
        const std::string src = E.emit_file(paper);
        std::ofstream f(out_path);
        if (!f) { snprintf(msg, msglen, "cannot write %s", out_path); return 3; }
        f << src; f.close();
        return 0;
    } catch (std::exception& e) { snprintf(msg, msglen, "%s", e.what()); return 3; }
}

// rank of a rational matrix, computed modulo a 61-bit prime (entries n/d -> n d^-1 mod p): never above the true rank and
// equal to it unless p divides one of the minors met on the way
static int rank_mod_p(const std::vector<Frac>& C, int m) {
    typedef unsigned long long u64; typedef unsigned __int128 u128;
    const u64 p = 2305843009213693951ull;      // 2^61 - 1
    auto mulm = [&](u64 a, u64 b) { return (u64)((u128)a * b % p); };
    auto powm = [&](u64 a, u64 e) { u64 r = 1; while (e) { if (e & 1) r = mulm(r, a); a = mulm(a, a); e >>= 1; } return r; };
    std::vector<u64> A((size_t)m * m);
    for (size_t i = 0; i < A.size(); ++i) {
        const long long nn = C[i].n, dd = C[i].d;
        const u64 an = (u64)((nn % (long long)p + (long long)p) % (long long)p);
        A[i] = mulm(an, powm((u64)(dd % (long long)p), p - 2));
    }
    int rank = 0;
    for (int col = 0; col < m && rank < m; ++col) {
        int piv = -1; for (int r = rank; r < m; ++r) if (A[(size_t)r * m + col]) { piv = r; break; }
        if (piv < 0) continue;
        for (int c = 0; c < m; ++c) std::swap(A[(size_t)piv * m + c], A[(size_t)rank * m + c]);
        const u64 inv = powm(A[(size_t)rank * m + col], p - 2);
        for (int r = rank + 1; r < m; ++r) {
            const u64 f = mulm(A[(size_t)r * m + col], inv);
            if (!f) continue;
            for (int c = col; c < m; ++c) A[(size_t)r * m + c] = (A[(size_t)r * m + c] + p - mulm(f, A[(size_t)rank * m + c])) % p;
        }
        ++rank;
    }
    return rank;
}

// The table program of a process for the generic kernels of csrc/device/heget_tab.cuh (no compilation needed).
// rc: 0 = ok, 1 = malformed process, 2 = unsupported / too large, 3 = internal error.  The caller owns the result.
heget::TabProgram* heget_build_table(const char* tag, const char* process, int* rc, char* msg, int msglen) {
    *rc = 3;
    try {
        Process P;
        try { P = parse_process(process); }
        catch (std::invalid_argument& e) { snprintf(msg, msglen, "%s", e.what()); *rc = 2; return 0; }
        catch (std::exception& e) { snprintf(msg, msglen, "%s", e.what()); *rc = 1; return 0; }
        if (P.n > 7) { snprintf(msg, msglen, "process with %d external legs is too large to build", P.n); *rc = 2; return 0; }
        int q = 0; for (int i = 0; i < P.n; ++i) q += P.legs[i].type != LEG_G;
        Graph G, GP; const Graph* paper = 0;
        try {
            G.merge = true; G.centroid = true; G.build(P, false);
            if (q == 4) { GP.build(P, true); paper = &GP; }
        } catch (std::exception& e) { snprintf(msg, msglen, "%s", e.what()); *rc = 2; return 0; }
        if (G.closings.empty()) { snprintf(msg, msglen, "process has no tree-level QCD diagram"); *rc = 2; return 0; }
        TabBuilder B(G, tag);
        { const char* f = getenv("HEGET_TAB_FOLD"); if (f && f[0] == '0') B.fold_parity = false; }      // HEGET_TAB_FOLD=0: evaluate both members of every parity pair
        B.build(paper);
        const Graph& GC = paper ? *paper : G;
        B.P.color_rank = rank_mod_p(GC.C, (int)GC.basis.size());
        *rc = 0;
        return new TabProgram(B.P);
    } catch (std::exception& e) { snprintf(msg, msglen, "%s", e.what()); return 0; }
}
