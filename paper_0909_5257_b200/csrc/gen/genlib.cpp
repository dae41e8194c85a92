// In-process entry to the process generator (step a0), used by
// heget_process_create when no pre-built plug-in exists for a process.  Same work as the hegetgen command line.
#include <cstdio>
#include <cstring>
#include <fstream>
#include "emit.hpp"

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
