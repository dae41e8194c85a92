// hegetgen: the host-side process generator of heget-b200.
//   hegetgen <tag> "<process>" <out.cu> [--block64 N] [--block32 N] [--jreg64 N] [--jreg32 N] [--share-closings 0|1]
// writes one specialised CUDA source for the process and prints a one-line summary (counts of Table 1).
//   hegetgen --summary "<process>"      prints the counts and the distinct colour-matrix values (Table 4)
#include <cstdio>
#include <cstring>
#include <fstream>
#include <set>
#include "emit.hpp"

using namespace heget;

static int two_lines(const Process& P) { int q = 0; for (int i = 0; i < P.n; ++i) q += P.legs[i].type != LEG_G; return q == 4; }

int main(int argc, char** argv) {
    try {
        if (argc >= 3 && !strcmp(argv[1], "--summary")) {
            Process P = parse_process(argv[2]);
            Graph G; G.build(P, true);
            std::set<std::pair<long long, long long> > vals;
            for (size_t i = 0; i < G.C.size(); ++i) if (!G.C[i].zero()) vals.insert(std::make_pair(G.C[i].n, G.C[i].d));
            printf("%s; diagrams %zu; topologies %d; colours %zu; distinct %zu;", argv[2], G.closings.size(), (int)std::lround(G.n_topologies), G.basis.size(), vals.size());
            for (std::set<std::pair<long long, long long> >::iterator it = vals.begin(); it != vals.end(); ++it) printf(" %lld/%lld", it->first, it->second);
            printf("\n");
            return 0;
        }
        if (argc < 4) { fprintf(stderr, "usage: hegetgen <tag> \"<process>\" <out.cu> [options]\n"); return 2; }
        EmitOptions opt; bool share = false;
        for (int i = 4; i + 1 < argc; i += 2) {
            if (!strcmp(argv[i], "--block64")) opt.block64 = atoi(argv[i + 1]);
            else if (!strcmp(argv[i], "--block32")) opt.block32 = atoi(argv[i + 1]);
            else if (!strcmp(argv[i], "--jreg64")) opt.jreg_max64 = atoi(argv[i + 1]);
            else if (!strcmp(argv[i], "--jreg32")) opt.jreg_max32 = atoi(argv[i + 1]);
            else if (!strcmp(argv[i], "--share-closings")) share = atoi(argv[i + 1]) != 0;
            else { fprintf(stderr, "unknown option %s\n", argv[i]); return 2; }
        }
        Process P = parse_process(argv[2]);
        // the kernel sums diagrams on the minimal (Fierzed) basis; for two quark lines the paper's over-complete
        // basis (reading A12) is built as well, for n_color and the colour matrix of Table 4
        Graph G; G.build(P, false);
        if (share) share_closings(G);      // experiment, off by default: fewer flops but 2x the live currents
        Graph GP; const Graph* paper = 0;
        if (two_lines(P)) { GP.build(P, true); paper = &GP; }
        Emitter E(G, argv[1], opt);
        std::string src = E.emit_file(paper);
        std::ofstream f(argv[3]); f << src; f.close();
        printf("%s: %zu diagrams, %d topologies, %zu colours (%zu evaluated, %d merged), %d/%d helicities, %zu ops, max %d live currents, %.0f flops/helicity, %d cache slots\n",
               argv[2], G.closings.size(), (int)std::lround(G.n_topologies), paper ? GP.basis.size() : G.basis.size(), G.basis.size(), E.NJ, E.NH, 1 << P.n,
               E.ops.size(), E.max_live, E.flops_hel, E.nslots);
        return 0;
    } catch (std::exception& e) { fprintf(stderr, "hegetgen: %s\n", e.what()); return 1; }
}
