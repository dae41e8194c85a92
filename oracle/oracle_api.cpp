// ORACLE (test infrastructure only): C entry points for tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs.  Nothing under paper_0909_5257_b200/ may use it.
//
// Momenta layout everywhere: SoA  mom[(leg*4 + mu)*n_events + e], legs in process-string order
// (two initial partons first), components (E, px, py, pz), GeV.
#include <cstdio>
#include <cstring>
#include <string>
#include <chrono>
#include <omp.h>
#include "su3.hpp"
#include "kin.hpp"
#include "rambo.hpp"
#include "diagrams.hpp"
#include "colour.hpp"
#include "eval.hpp"
#include "berends_giele.hpp"

using namespace orc;

static thread_local std::string g_err;

extern "C" {

const char* orc_last_error() { return g_err.c_str(); }

// keep_diagram_colour != 0 also stores every diagram's colour tensor (needed by tier O1)
void* orc_create(const char* process, double alpha_s, int keep_diagram_colour) {
    try {
        Model* M = new Model();
        Process P = parse_process(process);
        enumerate_diagrams(P, M->D);
        build_colour(M->D, M->cd, keep_diagram_colour != 0);
        M->gs = std::sqrt(4.0 * 3.14159265358979323846 * alpha_s);
        return M;
    } catch (std::exception& e) { g_err = e.what(); return 0; }
}
void orc_destroy(void* h) { delete (Model*)h; }

// info[0..]: n_ext, n_diagrams (paper convention), n_topologies, n_color, rank, n_pairings, n_nodes, n_assign
void orc_info(void* h, double* info) {
    Model* M = (Model*)h;
    info[0] = M->D.proc.n_ext(); info[1] = (double)M->D.diagrams.size(); info[2] = M->D.n_topologies;
    info[3] = M->cd.m; info[4] = M->cd.rank; info[5] = (double)M->D.pairings.size(); info[6] = (double)M->D.nodes.size();
    info[7] = (double)M->cd.n_assign;
    info[8] = M->D.proc.sym_factor; info[9] = M->D.proc.avg_color; info[10] = M->D.proc.avg_spin;
    info[11] = M->cd.C_max_imag; info[12] = M->cd.C_max_asym; info[13] = M->cd.max_residual;
    info[14] = M->cd.frac_nonzero_pairs; info[15] = M->cd.frac_all_zero; info[16] = M->gs;
}
void orc_colour_matrix(void* h, double* C) { Model* M = (Model*)h; std::memcpy(C, M->cd.C.data(), sizeof(double) * M->cd.C.size()); }
void orc_colour_eigenvalues(void* h, double* ev) { Model* M = (Model*)h; std::memcpy(ev, M->cd.eval.data(), sizeof(double) * M->cd.eval.size()); }

// legs of basis element alpha, flattened: kind, pairing, then 4 lists each preceded by its length
int orc_basis_element(void* h, int alpha, int* out) {
    Model* M = (Model*)h;
    const BasisElement& e = M->cd.basis[alpha];
    int n = 0; out[n++] = e.kind; out[n++] = e.pairing;
    for (int s = 0; s < 4; ++s) { out[n++] = (int)e.seq[s].size(); for (size_t i = 0; i < e.seq[s].size(); ++i) out[n++] = e.seq[s][i]; }
    return n;
}

void orc_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

void orc_sample_momenta(int n_final, double sqrt_s, double pt_min, double eta_max, double dr_min, uint64_t seed,
                        uint64_t first_event, uint64_t n_events, double* mom, double* weight, uint32_t* tries) {
    Cuts c; c.pt_min = pt_min; c.eta_max = eta_max; c.dr_min = dr_min;
    sample_momenta(n_final, sqrt_s, c, seed, first_event, n_events, mom, weight, tries);
}
int orc_pass_cuts(int n_final, const double* p_final /* [n][4] */, double pt_min, double eta_max, double dr_min) {
    Cuts c; c.pt_min = pt_min; c.eta_max = eta_max; c.dr_min = dr_min;
    return pass_cuts(n_final, (const double (*)[4])p_final, c) ? 1 : 0;
}
double orc_rambo_weight(int n_final, double sqrt_s) { return rambo_flat_weight(n_final, sqrt_s); }

static void gather(const double* mom, uint64_t n_events, uint64_t e, int n, double (*p)[4]) {
    for (int i = 0; i < n; ++i) for (int m = 0; m < 4; ++m) p[i][m] = mom[((size_t)i * 4 + m) * n_events + e];
}

// helicity-summed, colour-summed, averaged |M|^2 for n_events; tier 1 (needs keep_diagram_colour) or 2.
// n_threads <= 0: all cores.  Returns the seconds spent in the event loop.
double orc_me2(void* h, const double* mom, uint64_t n_events, int tier, int n_threads, double* out) {
    Model* M = (Model*)h;
    const int n = M->D.proc.n_ext();
    if (n_threads > 0) omp_set_num_threads(n_threads);
    auto t0 = std::chrono::steady_clock::now();
    #pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < (int64_t)n_events; ++e) {
        double p[16][4]; gather(mom, n_events, (uint64_t)e, n, p);
        out[e] = me2_event(*M, p, tier);
    }
    auto t1 = std::chrono::steady_clock::now();
    return std::chrono::duration<double>(t1 - t0).count();
}
int orc_max_threads() { return omp_get_max_threads(); }

// one event, one helicity configuration: colour-basis amplitudes J[2*m] (re,im), diagram amplitudes A[2*n_diag]
// (either may be NULL), returns sum_c |M^c|^2 (no averaging factors).  ward_leg >= 0: that gluon's eps -> p.
double orc_amplitudes(void* h, const double* p_aos /* [n_ext][4] */, const int* hel, int ward_leg, double* J_out, double* A_out) {
    Model* M = (Model*)h;
    std::vector<cplx> A, J;
    diagram_amplitudes(*M, (const double (*)[4])p_aos, hel, ward_leg, A);
    colour_amplitudes(*M, A, J);
    if (J_out) for (size_t i = 0; i < J.size(); ++i) { J_out[2 * i] = J[i].real(); J_out[2 * i + 1] = J[i].imag(); }
    if (A_out) for (size_t i = 0; i < A.size(); ++i) { A_out[2 * i] = A[i].real(); A_out[2 * i + 1] = A[i].imag(); }
    return colour_sum_O2(*M, J);
}
// same, colour sum by tier O1
double orc_colour_sum_O1(void* h, const double* p_aos, const int* hel) {
    Model* M = (Model*)h;
    std::vector<cplx> A;
    diagram_amplitudes(*M, (const double (*)[4])p_aos, hel, -1, A);
    return colour_sum_O1(*M, A);
}

// colour-ordered n-gluon partial amplitude by the Berends-Giele recursion (tier O3):
// order[n] = legs in trace order, all momenta/helicities PHYSICAL (as in orc_amplitudes); out[2] = (re, im)
void orc_bg_gluon(int n, const double* p_aos, const int* hel, const int* order, double gs, double* out) {
    cplx a = bg_partial_amplitude(n, (const double (*)[4])p_aos, hel, order, gs);
    out[0] = a.real(); out[1] = a.imag();
}
// colour-summed squared amplitude of one helicity configuration of an n-gluon process: explicit colour sum over Berends-Giele partial amplitudes
double orc_gluon_colour_sum_bg(int n, const double* p /* [n][4] */, const int* hel, double gs) {
    return gluon_colour_sum_bg(n, (const double (*)[4])p, hel, gs);
}

}  // extern "C"
